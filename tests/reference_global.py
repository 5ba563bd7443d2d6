"""Test-only helpers: the GLOBAL formulations the paper says AlgFAC must reproduce, written
with scipy on whole-level vectors.  Independent of oracle/ (different language, no composite
grids, no t/s accumulators) and of the CUDA path.

P:87  "the result obtained via the AlgFAC cycle should be exactly the same as that obtained by
       cycling on the entire grid while suppressing relaxation at certain points".
"""
import numpy as np
import scipy.sparse as sp


def l1_dinv(A):
    return 1.0 / np.asarray(abs(A).sum(axis=1)).ravel()


def masked_vcycles(As, Ps, masks, r0, niter, nu, cfs=None):
    """niter global V(nu,nu)-cycles (Alg. 1) on A_0 e = r0 from e = 0 in which level l
    relaxes only where masks[l] is True (l1-Jacobi, simultaneous update).  Returns e on level 0.
    cfs (list of +1/-1 arrays per level < L): "CF l1-scaled Jacobi" instead: every sweep is two
    half-sweeps, C-points then F-points before the coarse correction, F-points then C-points after it."""
    L = len(As) - 1
    dinv = [l1_dinv(A) for A in As]
    u = [np.zeros(A.shape[0]) for A in As]
    f = [np.array(r0, dtype=np.float64)] + [None] * L
    AL = As[L].toarray()

    def relax(l, first=+1):
        if cfs is None:
            d = dinv[l] * (f[l] - As[l] @ u[l])
            u[l][masks[l]] += d[masks[l]]
            return
        for cls in (first, -first):
            sel = masks[l] & ((cfs[l] > 0) == (cls > 0))
            d = dinv[l] * (f[l] - As[l] @ u[l])
            u[l][sel] += d[sel]

    for _ in range(niter):
        for l in range(L):
            if l != 0:
                u[l][:] = 0.0
            for _k in range(nu):
                relax(l)
            f[l + 1] = Ps[l].T @ (f[l] - As[l] @ u[l])
        u[L] = np.linalg.solve(AL, f[L])
        for l in range(L - 1, -1, -1):
            u[l] = u[l] + Ps[l] @ u[l + 1]
            for _k in range(nu):
                relax(l, -1)
    return u[0]


def hierarchy_from_oracle(o):
    As = [o.scipy_matrix(l, "A") for l in range(o.num_levels)]
    Ps = [o.scipy_matrix(l, "P") for l in range(o.num_levels - 1)]
    return As, Ps


def bfs_sets_bruteforce(A, seed, dist):
    """Points within graph distance <= dist of `seed` by all-pairs shortest paths (tiny graphs)."""
    from scipy.sparse.csgraph import shortest_path
    n = A.shape[0]
    G = sp.csr_matrix((np.ones(A.nnz), A.indices.copy(), A.indptr.copy()), shape=A.shape)
    G.setdiag(0)
    G.eliminate_zeros()
    D = shortest_path(G, method="FW", directed=True, unweighted=True)
    d = D[np.asarray(seed, dtype=np.int64), :].min(axis=0)
    return np.nonzero(d <= dist)[0]


def resum_galerkin_two_stage(o):
    """Turn the oracle object `o` into a SECOND valid oracle under reading S4 (the terms of a Galerkin entry may be summed in
    any order): every coarse operator is replaced, level by level, by scipy's two-stage product P_l^T (A_l P_l) of the
    oracle's own P_l and its (already replaced) A_l, scattered onto the stored pattern (what scipy drops as an exact zero
    stays 0.0).  Nothing of the CUDA path enters.  The new values differ from the one-pass triple loop of the oracle's
    `galerkin` by rounding only; returns the largest entry change per level relative to the largest entry."""
    moved = []
    for l in range(o.num_levels - 1):
        A, P = o.scipy_matrix(l, "A"), o.scipy_matrix(l, "P")
        C = (P.T.tocsr() @ (A @ P)).tocsr()
        C.sort_indices()
        rp, ci, v = o.matrix(l + 1, "A")
        n = len(rp) - 1
        key = np.repeat(np.arange(n, dtype=np.int64), np.diff(rp)) * n + ci       # ascending: rows have ascending columns
        ckey = np.repeat(np.arange(n, dtype=np.int64), np.diff(C.indptr)) * n + C.indices
        pos = np.searchsorted(key, ckey)
        assert (pos < len(key)).all() and (key[pos] == ckey).all(), "scipy's product has an entry outside the oracle's pattern"
        nv = np.zeros_like(v)
        nv[pos] = C.data
        moved.append(float(np.abs(nv - v).max() / np.abs(v).max()))
        o.set_level_values(l + 1, nv)
    return moved
