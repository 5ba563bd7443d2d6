"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Every test names the passage (P:NNN = PAPER.md line) or the SURVEY.md §8(c) reading it pins.
None of them re-types the oracle's formulas in the oracle's own structure: they use closed
forms, brute force on tiny inputs, scipy/numpy library routines on whole-level (global)
vectors, or invariants.
"""
import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spla

import workloads as wl
from oracle import Oracle
from tests.reference_global import (bfs_sets_bruteforce, hierarchy_from_oracle, l1_dinv,
                                    masked_vcycles)


def make_oracle(p, **kw):
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, kw.get("theta", p.theta), kw.get("max_levels", p.max_levels),
               kw.get("coarse_max", p.coarse_max))
    o.set_partition(p.num_subdomains, p.owner, kw.get("eta", p.eta), kw.get("num_ghost", p.num_ghost))
    return o


# ------------------------------------------------------------------------------------------
# input generator
# ------------------------------------------------------------------------------------------
def test_mt19937_64_known_answer():
    # ISO C++ [rand.predef]: the 10000th invocation of a default-constructed mt19937_64
    # (seed 5489) produces 9981545732273789042.
    assert int(wl.raw_draws(5489, 10000)[-1]) == 9981545732273789042
    u = wl.uniform(7, 1000)
    assert (u >= 0).all() and (u < 1).all()


def test_config_sizes_match_baseline():
    # BASELINE.json configs: N and nnz of configs 1 and 2
    p1 = wl.make_config(1)
    assert (p1.n, p1.nnz, p1.num_subdomains) == (1089, 5313, 4)
    p2 = wl.make_config(2)
    assert (p2.n, p2.nnz, p2.num_subdomains) == (262144, 1810432, 64)
    assert np.bincount(p2.owner).tolist() == [4096] * 64


# ------------------------------------------------------------------------------------------
# S1-S4: 1D Poisson closed form.  tridiag(-1,2,-1), n = 2^k - 1: C = odd indices on every level,
# interpolation weights 1/2, and A_l = 2^-l tridiag(-1,2,-1) bit-exactly.
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [4, 6])
def test_1d_poisson_hierarchy_closed_form(k):
    n = 2 ** k - 1
    rp, ci, v = wl.poisson1d(n)
    o = Oracle(n, rp, ci, v, 0.25, 25, 1)
    assert o.num_levels == k
    for l in range(o.num_levels):
        nl = 2 ** (k - l) - 1
        assert o.level_size(l)[0] == nl
        A = o.scipy_matrix(l, "A").toarray()
        T = (2.0 * np.eye(nl) - np.eye(nl, k=1) - np.eye(nl, k=-1)) * 2.0 ** (-l)
        assert np.array_equal(A, T)
        if l < o.num_levels - 1:
            cf = o.cf(l)
            assert np.array_equal(np.nonzero(cf == 1)[0], np.arange(1, nl, 2))
            P = o.scipy_matrix(l, "P").toarray()
            Pref = np.zeros((nl, (nl - 1) // 2))
            for c in range((nl - 1) // 2):
                Pref[2 * c + 1, c] = 1.0
                Pref[2 * c, c] = 0.5
                Pref[2 * c + 2, c] = 0.5
            assert np.array_equal(P, Pref)


def _strength_bruteforce(A, theta):
    """S1 literally, dense."""
    n = A.shape[0]
    M = A.toarray()
    pat = sp.csr_matrix((np.ones(A.nnz), A.indices, A.indptr), shape=A.shape).toarray() > 0
    S = np.zeros((n, n), dtype=bool)
    for i in range(n):
        offs = [k for k in range(n) if k != i and pat[i, k]]
        if not offs:
            continue
        m = max(-M[i, k] for k in offs)
        if m <= 0:
            continue
        for j in offs:
            if -M[i, j] > 0 and -M[i, j] >= theta * m * (1 - 1e-10):
                S[i, j] = True
    return S


def _rs_first_pass_bruteforce(S):
    """S2 by linear scans (O(n^2)): undecided point of largest lambda, ties to the smallest index."""
    n = S.shape[0]
    lam = S.sum(axis=0).astype(int)           # |S_i^T|
    cf = np.zeros(n, dtype=int)
    for i in range(n):
        if not S[i].any() and lam[i] == 0:
            cf[i] = -1
    while (cf == 0).any():
        und = np.nonzero(cf == 0)[0]
        i = und[np.argmax(lam[und])]          # argmax returns the first (smallest index) maximum
        cf[i] = 1
        for j in np.nonzero(S[:, i])[0]:
            if cf[j] == 0:
                cf[j] = -1
                for k in np.nonzero(S[j])[0]:
                    if cf[k] == 0:
                        lam[k] += 1
    return cf


@pytest.mark.parametrize("cfg,scale,theta", [(1, 9, 0.25), (4, 5, 0.5), (5, 12, 0.25), (3, 4, 0.5), (6, 10, 0.25)])
def test_strength_and_cf_split_bruteforce(cfg, scale, theta):
    p = wl.make_config(cfg, scale)
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, theta, 3, 4)
    for l in range(o.num_levels - 1):
        A = o.scipy_matrix(l, "A")
        S = _strength_bruteforce(A, theta)
        cf = _rs_first_pass_bruteforce(S)
        assert np.array_equal(cf, o.cf(l).astype(int)), f"level {l}"
        # invariants of the first pass: every F-point with strong connections has a strong C
        # neighbour it depends on OR was never reached; no C-point strongly depends on an
        # earlier C-point.  With symmetric strength: C is independent in the strength graph.
        if np.array_equal(S, S.T):
            C = cf == 1
            assert not S[np.ix_(C, C)].any()


def test_direct_interpolation_rows():
    # S3: C rows are injection; F rows with zero row sum interpolate constants exactly
    # (sum_j w_ij = -sum_neg / (a_ii + sum_pos) = 1 when the row sums to zero).
    p = wl.make_config(4, 8)
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, 0.5, 25, 8)
    A = o.scipy_matrix(0, "A")
    P = o.scipy_matrix(0, "P")
    cf = o.cf(0)
    rowsum = np.asarray(A.sum(axis=1)).ravel()
    prow = np.asarray(P.sum(axis=1)).ravel()
    cidx = np.cumsum(cf == 1) - 1
    for i in np.nonzero(cf == 1)[0]:
        assert P.indices[P.indptr[i]:P.indptr[i + 1]].tolist() == [cidx[i]]
        assert P.data[P.indptr[i]] == 1.0
    interior = (np.abs(rowsum) < 1e-12 * A.diagonal()) & (cf == -1) & (np.diff(P.indptr) > 0)
    assert interior.sum() > 10
    assert np.allclose(prow[interior], 1.0, rtol=0, atol=1e-13)
    # weights are proportional to the strong C entries of the row: w_ij / a_ij constant per row
    for i in np.nonzero(interior)[0][:20]:
        cols = P.indices[P.indptr[i]:P.indptr[i + 1]]
        fine = np.nonzero(cf == 1)[0][cols]
        ratio = P.data[P.indptr[i]:P.indptr[i + 1]] / np.asarray(A[i, fine].todense()).ravel()
        assert np.allclose(ratio, ratio[0], rtol=1e-13)
        assert (ratio < 0).all()          # a_ij < 0, w_ij > 0


def test_direct_interpolation_with_positive_offdiagonals():
    # S3 / reading A11 on the paper's Problem 2 (rotated anisotropy, bilinear FE: some off-diagonals are
    # positive): w_ij = -alpha_i a_ij / d_i with d_i = a_ii + sum of the positive off-diagonals,
    # alpha_i = (sum of the negative off-diagonals) / (sum over the strong C neighbours), written out with numpy
    p = wl.make_config(6, 12)
    theta = 0.25
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, theta, 25, 8)
    A = o.scipy_matrix(0, "A").toarray()
    assert ((A - np.diag(np.diag(A))) > 0).sum() > 100
    P = o.scipy_matrix(0, "P").toarray()
    cf = o.cf(0)
    cidx = np.cumsum(cf == 1) - 1
    checked = 0
    for i in np.nonzero(cf == -1)[0]:
        off = A[i].copy(); off[i] = 0.0
        nz = off != 0
        m = (-off[nz]).max() if nz.any() else 0.0
        strong = (off != 0) & (-off > 0) & (-off >= theta * m * (1 - 1e-10))
        Ci = np.nonzero(strong & (cf == 1))[0]
        if len(Ci) == 0:
            assert not P[i].any()
            continue
        d = A[i, i] + off[off > 0].sum()
        alpha = off[off < 0].sum() / off[Ci].sum()
        w = np.zeros(P.shape[1])
        w[cidx[Ci]] = -alpha * off[Ci] / d
        assert np.allclose(P[i], w, rtol=1e-13, atol=1e-15), i
        checked += 1
    assert checked > 30


@pytest.mark.parametrize("cfg,scale", [(2, 8), (3, 6), (4, 6), (5, 16), (6, 12)])
def test_galerkin_matches_library_triple_product(cfg, scale):
    # S4 / P:49: A_{l+1} = R_l A_l P_l with R_l = P_l^T; every structural entry kept.
    p = wl.make_config(cfg, scale)
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, p.theta, 25, 8)
    assert o.num_levels >= 3
    for l in range(o.num_levels - 1):
        A, P, Ac = o.scipy_matrix(l, "A"), o.scipy_matrix(l, "P"), o.scipy_matrix(l + 1, "A")
        ref = (P.T @ A @ P).toarray()
        assert np.allclose(Ac.toarray(), ref, rtol=1e-13, atol=1e-14 * abs(ref).max())
        # structural pattern = boolean product of the patterns
        pat = lambda M: sp.csr_matrix((np.ones(M.nnz), M.indices, M.indptr), shape=M.shape)
        bref = (pat(P).T @ pat(A) @ pat(P)).toarray() > 0
        got = pat(Ac).toarray() > 0
        assert np.array_equal(got, bref)
        assert np.allclose(Ac.toarray(), Ac.toarray().T, rtol=1e-12, atol=1e-14)
        # columns strictly ascending
        for i in range(Ac.shape[0]):
            c = Ac.indices[Ac.indptr[i]:Ac.indptr[i + 1]]
            assert (np.diff(c) > 0).all()


def test_fe27_stored_zero_faces_are_edges():
    # A8: a stored entry is an edge whatever its value (the 27-point FE stencil has exact zeros)
    p = wl.make_config(3, 6)
    assert (p.vals == 0.0).sum() > 0
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, 0.5, 2, 4)
    o.set_partition(1, np.zeros(p.n, np.int32), 0, 1)
    # one subdomain owning everything: trivial; use a 2-subdomain split instead
    own = (np.arange(p.n) % 6 >= 3).astype(np.int32)
    o.set_partition(2, own, 0, 1)
    real, ghost = o.composite(0, 0)
    A = o.scipy_matrix(0, "A")
    # ghost of eta=0: all stored neighbours of owned points, including the zero-valued faces
    x = np.arange(p.n) % 6
    face_nb = np.nonzero((own == 1) & (x == 3))[0]
    assert np.isin(face_nb, ghost).all()


def test_l1_diagonal():
    # S8 / reading A2: D_ii = sum_j |a_ij| over the full row
    p = wl.make_config(4, 6)
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, 0.5, 25, 8)
    for l in range(o.num_levels):
        A = o.scipy_matrix(l, "A")
        assert np.allclose(o.dinv(l), l1_dinv(A), rtol=1e-14)


def test_dense_coarse_solve_matches_library():
    p = wl.make_config(1)
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, 0.25, 25, 16)
    AL = o.scipy_matrix(o.num_levels - 1, "A").toarray()
    rhs = wl.rhs(11, AL.shape[0])
    assert np.allclose(o.coarse_solve(rhs), np.linalg.solve(AL, rhs), rtol=1e-12)


# ------------------------------------------------------------------------------------------
# S6/S7 composite sets by brute force (eq. 1)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,scale,parts,eta,ng", [(1, 13, 2, 1, 1), (1, 13, 3, 2, 1), (1, 11, 2, 0, 2),
                                                    (2, 6, 2, 1, 1), (5, 14, 2, 3, 1), (3, 5, 2, 1, 1)])
def test_composite_sets_bruteforce(cfg, scale, parts, eta, ng):
    p = wl.make_config(cfg, scale, parts_per_dim=parts)
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, p.theta, 25, 6)
    o.set_partition(p.num_subdomains, p.owner, eta, ng)
    L = o.num_levels - 1
    As = [o.scipy_matrix(l, "A") for l in range(o.num_levels)]
    union = np.zeros(p.n, dtype=int)
    for q in range(p.num_subdomains):
        B = np.nonzero(p.owner == q)[0]
        union[B] += 1
        for l in range(o.num_levels):
            real, ghost = o.composite(q, l)
            if l == L:
                assert np.array_equal(real, np.arange(As[l].shape[0]))     # A5
                assert len(ghost) == 0
                break
            D = bfs_sets_bruteforce(As[l], B, eta)
            Dbar = bfs_sets_bruteforce(As[l], D, ng)
            assert np.array_equal(real, D), (q, l)
            assert np.array_equal(ghost, np.setdiff1d(Dbar, D)), (q, l)
            if l == 0:
                assert np.isin(B, real).all()
            # eq. 1: every stored column of a real row lies in D-bar_l
            A = As[l]
            for i in real:
                assert np.isin(A.indices[A.indptr[i]:A.indptr[i + 1]], Dbar).all()
            cf = o.cf(l)
            cidx = np.cumsum(cf == 1) - 1
            B = cidx[D[cf[D] == 1]]
    assert (union == 1).all()                                          # owned sets partition Omega_0


def test_large_eta_gives_whole_levels():
    p = wl.make_config(1, 13)
    o = make_oracle(p, eta=50, coarse_max=6)
    for q in range(4):
        for l in range(o.num_levels):
            real, ghost = o.composite(q, l)
            assert len(real) == o.level_size(l)[0] and len(ghost) == 0


# ------------------------------------------------------------------------------------------
# Alg. 4 against the global formulation and special cases
# ------------------------------------------------------------------------------------------
def _masks(o, q):
    masks = []
    for l in range(o.num_levels):
        m = np.zeros(o.level_size(l)[0], dtype=bool)
        m[o.composite(q, l)[0]] = True
        masks.append(m)
    return masks


@pytest.mark.parametrize("cfg,scale,parts,eta,nfac,nu", [
    (1, None, 2, 1, 1, 1), (1, None, 2, 1, 2, 1), (1, None, 2, 1, 3, 2), (1, 21, 3, 2, 2, 1),
    (2, 12, 2, 2, 2, 1), (2, 12, 2, 1, 3, 2), (4, 12, 2, 2, 2, 1), (5, 32, 2, 3, 2, 1), (3, 8, 2, 1, 2, 1), (6, 32, 2, 1, 2, 1)])
def test_algfac_equals_masked_global_vcycle(cfg, scale, parts, eta, nfac, nu):
    # P:87 guiding principle; eqs. 13-30; Alg. 4
    p = wl.make_config(cfg, scale, parts_per_dim=parts)
    o = make_oracle(p, eta=eta, coarse_max=min(p.coarse_max, 16))
    assert o.num_levels >= 3
    As, Ps = hierarchy_from_oracle(o)
    r0 = wl.rhs(123, p.n)
    for q in range(p.num_subdomains):
        real, ghost = o.composite(q, 0)
        u_fac = o.fac_local(q, r0, nfac, nu)
        assert o.dropped() == 0                                        # A7
        u_glob = masked_vcycles(As, Ps, _masks(o, q), r0, nfac, nu)
        idx = np.concatenate([real, ghost])
        scale_ = np.abs(u_glob).max()
        tol = 1e-12 if cfg == 5 else 1e-13          # config 5: 1e4 coefficient jumps, cond(A_l) ~ 1e7
        assert np.abs(u_fac - u_glob[idx]).max() <= tol * scale_, (q,)


@pytest.mark.parametrize("nu", [1, 2])
def test_single_subdomain_is_plain_vcycle(nu):
    # north_star: one subdomain whose padding covers the whole domain => one FAC cycle equals a
    # standard AMG V(nu,nu)-cycle (Alg. 1) with the same relaxation.
    p = wl.make_config(1, 21, parts_per_dim=1)
    o = make_oracle(p, eta=100, coarse_max=8)
    As, Ps = hierarchy_from_oracle(o)
    r0 = wl.rhs(5, p.n)
    all_true = [np.ones(A.shape[0], dtype=bool) for A in As]
    u_v = masked_vcycles(As, Ps, all_true, r0, 1, nu)
    u_fac = o.fac_local(0, r0, 1, nu)
    assert np.abs(u_fac - u_v).max() <= 1e-13 * np.abs(u_v).max()
    # the oracle's own Alg. 1 agrees as well, and so does a whole AMG-DD cycle from x = 0
    u_alg1 = o.vcycle(r0, np.zeros(p.n), nu, nu)
    assert np.abs(u_alg1 - u_v).max() <= 1e-13 * np.abs(u_v).max()
    x = np.zeros(p.n)
    o.cycle(r0, x, 1, nu)
    assert np.abs(x - u_v).max() <= 1e-13 * np.abs(u_v).max()


# ------------------------------------------------------------------------------------------
# CF l1-Jacobi (reading A2b)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,scale,parts,eta,nfac,nu", [
    (1, None, 2, 1, 2, 1), (1, 21, 3, 2, 3, 2), (2, 12, 2, 2, 2, 1), (4, 12, 2, 2, 2, 2), (5, 32, 2, 3, 2, 1), (3, 8, 2, 1, 2, 1)])
def test_cf_jacobi_algfac_equals_masked_global_vcycle(cfg, scale, parts, eta, nfac, nu):
    # the P:87 equivalence holds for any point-wise relaxation: here C- then F-points before, F- then
    # C-points after the coarse correction; the global formulation is scipy code of its own
    p = wl.make_config(cfg, scale, parts_per_dim=parts)
    o = make_oracle(p, eta=eta, coarse_max=min(p.coarse_max, 16))
    o.set_smoother(1)
    As, Ps = hierarchy_from_oracle(o)
    cfs = [o.cf(l) for l in range(o.num_levels - 1)]
    r0 = wl.rhs(321, p.n)
    for q in range(p.num_subdomains):
        real, ghost = o.composite(q, 0)
        u_fac = o.fac_local(q, r0, nfac, nu)
        u_glob = masked_vcycles(As, Ps, _masks(o, q), r0, nfac, nu, cfs=cfs)
        idx = np.concatenate([real, ghost])
        tol = 1e-12 if cfg == 5 else 1e-13
        assert np.abs(u_fac - u_glob[idx]).max() <= tol * np.abs(u_glob).max(), (q,)
    # it is a different method from plain l1-Jacobi
    u_cf = o.fac_local(0, r0, nfac, nu)
    o.set_smoother(0)
    assert np.abs(o.fac_local(0, r0, nfac, nu) - u_cf).max() > 1e-6 * np.abs(u_cf).max()


def test_cf_jacobi_half_sweeps():
    # one sweep = (I - M_F D^-1 A)(I - M_C D^-1 A) on the error, written with dense matrices: C-points first
    p = wl.make_config(1, 9, parts_per_dim=1)
    o = make_oracle(p, eta=100, coarse_max=4)
    o.set_smoother(1)
    A = o.scipy_matrix(0, "A").toarray()
    cf = o.cf(0)
    Dinv = np.diag(1.0 / np.abs(A).sum(axis=1))
    MC, MF = np.diag((cf > 0).astype(float)), np.diag((cf < 0).astype(float))
    rng = np.random.default_rng(0)
    u, f = rng.standard_normal(p.n), rng.standard_normal(p.n)
    u1 = u + MC @ Dinv @ (f - A @ u)
    u2 = u1 + MF @ Dinv @ (f - A @ u1)
    assert np.abs(o.relax(0, u, f) - u2).max() <= 1e-14 * np.abs(u2).max()
    # all points in one class: plain l1-Jacobi; and the V-cycle of Alg. 1 uses the same relaxation
    o.set_smoother(0)
    assert np.abs(o.relax(0, u, f) - (u + Dinv @ (f - A @ u))).max() <= 1e-14 * np.abs(u).max()
    o.set_smoother(1)
    As, Ps = hierarchy_from_oracle(o)
    cfs = [o.cf(l) for l in range(o.num_levels - 1)]
    all_true = [np.ones(M.shape[0], dtype=bool) for M in As]
    u_v = masked_vcycles(As, Ps, all_true, f, 1, 1, cfs=cfs)
    assert np.abs(o.vcycle(f, np.zeros(p.n), 1, 1) - u_v).max() <= 1e-13 * np.abs(u_v).max()
    # C-points are relaxed exactly once per half sweep: after the C half the residual of a C-row whose
    # neighbours are all F-points changes only through its own update (1D-like check on the diagonal scaling)
    r_before = f - A @ u
    r_after = f - A @ u1
    i = int(np.nonzero(cf > 0)[0][0])
    nbrs = np.nonzero(A[i])[0]
    if all(cf[j] < 0 for j in nbrs if j != i):
        assert np.isclose(r_after[i], r_before[i] * (1.0 - A[i, i] * Dinv[i, i]), rtol=1e-12)


def test_num_ghost_invariance():
    # A13: extra ghost layers are stored and interpolated but never read by a real row
    p = wl.make_config(1)
    xs = []
    for ng in (1, 2, 3):
        o = make_oracle(p, num_ghost=ng)
        x = np.zeros(p.n)
        o.solve(p.b, x, 2, 2, 1)
        xs.append(x)
    assert np.abs(xs[0] - xs[1]).max() <= 1e-15 * np.abs(xs[0]).max()
    assert np.abs(xs[0] - xs[2]).max() <= 1e-15 * np.abs(xs[0]).max()


# ------------------------------------------------------------------------------------------
# relaxation: closed-form Jacobi eigenvalues (SURVEY.md §8(c) pins table)
# ------------------------------------------------------------------------------------------
def test_jacobi_eigenvalues_1d():
    # error operator I - D^{-1}A with D = 4 I on tridiag(-1,2,-1): eigenvector sin(k pi j/(n+1)),
    # eigenvalue 1 - (2 - 2 cos(k pi h))/4 = cos^2(k pi h / 2); smoothing factor 1/2.
    n = 31
    rp, ci, v = wl.poisson1d(n)
    o = Oracle(n, rp, ci, v, 0.25, 1, 1)
    j = np.arange(1, n + 1)
    h = 1.0 / (n + 1)
    worst_high = 0.0
    for k in range(1, n + 1):
        e = np.sin(k * np.pi * j * h)
        e1 = o.relax(0, e, np.zeros(n), dinv=np.full(n, 0.25))
        lam = np.cos(k * np.pi * h / 2) ** 2
        assert np.allclose(e1, lam * e, rtol=0, atol=1e-14)
        if k >= (n + 1) // 2:
            worst_high = max(worst_high, lam)
    assert abs(worst_high - 0.5) < 1e-12
    # S8 proper: l1 value is 4 in the interior and 3 at the two Dirichlet-adjacent rows
    d = 1.0 / o.dinv(0)
    assert d[0] == 3.0 and d[-1] == 3.0 and (d[1:-1] == 4.0).all()


def test_jacobi_eigenvalues_2d():
    # D = 8 I on the 5-point Laplacian: eigenvalue (cos^2(k pi h/2) + cos^2(m pi h/2))/2;
    # smoothing factor 3/4 (worst high-frequency mode k = n, m -> 1 ... here bounded by 3/4).
    n = 15
    rp, ci, v = wl.poisson2d_5pt(n)
    o = Oracle(n * n, rp, ci, v, 0.25, 1, 1)
    h = 1.0 / (n + 1)
    jx, jy = np.meshgrid(np.arange(1, n + 1), np.arange(1, n + 1), indexing="xy")
    worst = 0.0
    for k in (1, 3, 8, 15):
        for m in (1, 2, 8, 15):
            e = (np.sin(k * np.pi * jx * h) * np.sin(m * np.pi * jy * h)).ravel()
            e2 = o.relax(0, e, np.zeros(n * n), dinv=np.full(n * n, 0.125), nsweeps=2)
            lam = (np.cos(k * np.pi * h / 2) ** 2 + np.cos(m * np.pi * h / 2) ** 2) / 2
            assert np.allclose(e2, lam ** 2 * e, rtol=0, atol=1e-14)
            if max(k, m) >= (n + 1) // 2:
                worst = max(worst, lam)
    assert worst < 0.75 + 1e-12


def test_relax_mask_only_touches_real_points():
    # ghost points are not relaxed
    p = wl.make_config(1, 9)
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, 0.25, 1, 1)
    mask = (np.arange(p.n) % 3 == 0).astype(np.int8)
    u = wl.rhs(3, p.n)
    f = wl.rhs(4, p.n)
    A = o.scipy_matrix(0, "A")
    u1 = o.relax(0, u, f, mask=mask)
    ref = u + l1_dinv(A) * (f - A @ u)
    assert np.array_equal(u1[mask == 0], u[mask == 0])
    assert np.allclose(u1[mask == 1], ref[mask == 1], rtol=1e-14, atol=1e-15)


# ------------------------------------------------------------------------------------------
# Alg. 2 with several subdomains: the owned-correction update
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,scale,parts,eta,nfac,nu", [(1, None, 2, 1, 2, 1), (1, 21, 3, 2, 1, 2), (2, 12, 2, 2, 2, 1),
                                                         (4, 12, 2, 2, 2, 1), (5, 32, 2, 3, 2, 1)])
def test_cycle_with_several_subdomains_is_the_patchwork_of_local_solves(cfg, scale, parts, eta, nfac, nu):
    """Alg. 2 for P > 1, against a restatement that uses nothing of the oracle's cycle driver:
    r = b - A_0 x (scipy); for every p the global V-cycles with relaxation masked to D_l^p (scipy, whole-level
    vectors) give e^p; the new iterate is x + e^p ON Omega_0^p ONLY ("each processor updates only its owned dofs",
    P:65).  Starts from a nonzero x so that the residual line P:471 matters, checks every dof, and checks
    that a partial list of subdomains leaves every other dof bit-identical."""
    p = wl.make_config(cfg, scale, parts_per_dim=parts)
    assert p.num_subdomains > 1
    o = make_oracle(p, eta=eta, coarse_max=min(p.coarse_max, 16))
    As, Ps = hierarchy_from_oracle(o)
    A = sp.csr_matrix((p.vals, p.colind, p.rowptr), shape=(p.n, p.n))
    x0 = 0.1 * wl.rhs(77, p.n)
    r0 = p.b - A @ x0
    expect = x0.copy()
    for q in range(p.num_subdomains):
        e = masked_vcycles(As, Ps, _masks(o, q), r0, nfac, nu)
        own = p.owner == q
        expect[own] = x0[own] + e[own]
    x = x0.copy()
    o.cycle(p.b, x, nfac, nu)
    tol = 1e-12 if cfg == 5 else 1e-13
    assert np.abs(x - expect).max() <= tol * np.abs(expect).max()
    # a subset of the subdomains: only their owned dofs move, the others keep their bits
    some = np.array([0, p.num_subdomains - 1], dtype=np.int32)
    x2 = x0.copy()
    o.cycle(p.b, x2, nfac, nu, subdomains=some)
    moved = np.isin(p.owner, some)
    assert np.array_equal(x2[~moved], x0[~moved])
    assert np.array_equal(x2[moved], x[moved])
    # and the oracle's own per-subdomain routine composes to the same thing (the composition the GPU tests rely on)
    x3 = x0.copy()
    for q in range(p.num_subdomains):
        real, _ = o.composite(q, 0)
        u0 = o.fac_local(q, r0, nfac, nu)
        own_local = p.owner[real] == q
        x3[real[own_local]] += u0[:len(real)][own_local]
    assert np.array_equal(x3, x)


# ------------------------------------------------------------------------------------------
# a8 with row exchanges (Alg. 4; "a direct method")
# ------------------------------------------------------------------------------------------
def test_dense_coarse_solve_with_row_exchanges():
    rp, ci, v, dense = wl.pivoting_band_matrix()
    n = dense.shape[0]
    assert np.linalg.cond(dense) < 1e6
    # partial pivoting must actually exchange rows here: scipy's LU of the same matrix is not the identity permutation
    import scipy.linalg as sla
    _, piv = sla.lu_factor(dense)
    assert (piv != np.arange(n)).sum() >= n // 2
    o = Oracle(n, rp, ci, v, 0.25, 25, n)                    # coarse_max >= n: L = 0, A_L = A_0 (S5)
    assert o.num_levels == 1
    for seed in (1, 2, 3):
        rhs = wl.rhs(seed, n)
        sol = np.linalg.solve(dense, rhs)
        assert np.abs(o.coarse_solve(rhs) - sol).max() <= 1e-11 * np.abs(sol).max()
    # through Alg. 2 / Alg. 4 with L = 0 (reading A5): one cycle is the direct solve, whatever the partition
    owner = (np.arange(n) * 3 // n).astype(np.int32)
    o.set_partition(3, owner, 1, 1)
    b = wl.rhs(9, n)
    x = np.zeros(n)
    o.cycle(b, x, 1, 1)
    sol = np.linalg.solve(dense, b)
    assert np.abs(x - sol).max() <= 1e-11 * np.abs(sol).max()


# ------------------------------------------------------------------------------------------
# whole solve
# ------------------------------------------------------------------------------------------
def test_solve_converges_to_direct_solution():
    p = wl.make_config(1, 9, parts_per_dim=2)
    o = make_oracle(p, coarse_max=4)
    x = np.zeros(p.n)
    res = o.solve(p.b, x, 60, 2, 1)
    A = sp.csr_matrix((p.vals, p.colind, p.rowptr), shape=(p.n, p.n))
    xd = spla.spsolve(A.tocsc(), p.b)
    assert np.abs(x - xd).max() <= 1e-14 * np.abs(xd).max() + 1e-15
    assert res[-1] < 1e-13 * res[0]


@pytest.mark.parametrize("cfg,scale,parts", [(1, None, 2), (2, 16, 2), (4, 12, 2)])
def test_residual_monotone_and_norm_definition(cfg, scale, parts):
    # north_star: residual reduction must be monotone (configs 1-4); A16: plain 2-norm of b - A x
    p = wl.make_config(cfg, scale, parts_per_dim=parts)
    o = make_oracle(p)
    x = np.zeros(p.n)
    res = o.solve(p.b, x, 6, 2, 1)
    assert (np.diff(res) < 0).all()
    A = sp.csr_matrix((p.vals, p.colind, p.rowptr), shape=(p.n, p.n))
    assert np.isclose(res[0], np.linalg.norm(p.b), rtol=1e-14)
    assert np.isclose(res[-1], np.linalg.norm(p.b - A @ x), rtol=1e-9)


def test_config1_convergence_range():
    # orientation only: config 1 drops by roughly 0.05-0.12 per cycle
    p = wl.make_config(1)
    o = make_oracle(p)
    x = np.zeros(p.n)
    res = o.solve(p.b, x, 3, 2, 1)
    rho = res[1:] / res[:-1]
    assert (rho > 0.02).all() and (rho < 0.2).all()


def test_matvec_counts():
    # a V(nu1,nu2)-cycle costs (1+nu1+nu2) A-matvecs + one P + one R per level.
    # AlgFAC adds one A_{l+1}-matvec per coarse level, absent on the initial downsweep.
    p = wl.make_config(1)
    o = make_oracle(p)
    L = o.num_levels - 1
    r0 = p.b
    for nfac, nu in [(1, 1), (2, 1), (3, 2)]:
        o.fac_local(0, r0, nfac, nu)
        c = o.counters()
        assert c["A"] == nfac * L * (1 + 2 * nu) + (nfac - 1) * L
        assert c["P"] == nfac * L and c["R"] == nfac * L


def test_overhead_definition():
    # sum over composite grids and levels of nnz(A_l) on real rows / sum_l nnz(A_l)
    p = wl.make_config(1)
    o = make_oracle(p)
    num = 0
    den = 0
    for l in range(o.num_levels):
        A = o.scipy_matrix(l, "A")
        den += A.nnz
        for q in range(4):
            real, _ = o.composite(q, l)
            num += np.diff(A.indptr)[real].sum()
    assert np.isclose(o.overhead(), num / den, rtol=1e-14)
    # one subdomain covering everything has overhead exactly 1
    p1 = wl.make_config(1, parts_per_dim=1)
    assert make_oracle(p1, eta=100).overhead() == 1.0


# ------------------------------------------------------------------------------------------
# stored values (tests/golden/, written by tests/golden/make_golden.py from oracle/ only)
# ------------------------------------------------------------------------------------------
def _golden(name):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    return np.array([float(ln) for ln in open(path) if not ln.startswith("#")])


@pytest.mark.parametrize("name,cfg,scale,smoother", [("config1_resnorms.txt", 1, None, 0), ("config4_scale24_resnorms.txt", 4, 24, 0),
                                                      ("config1_cfjacobi_resnorms.txt", 1, None, 1)])
def test_oracle_reproduces_stored_residual_norms(name, cfg, scale, smoother):
    p = wl.make_config(cfg, scale)
    o = make_oracle(p)
    o.set_smoother(smoother)
    res = o.solve(p.b, np.zeros(p.n), p.num_cycles, p.num_fac_cycles, p.relax_sweeps)
    ref = _golden(name)
    assert len(ref) == p.num_cycles + 1
    assert np.allclose(res, ref, rtol=1e-12, atol=0), (res, ref)        # thread count / summation order of the oracle's host may differ in the last digits
    assert res[0] == pytest.approx(np.linalg.norm(p.b), rel=1e-14)      # k = 0: x = 0 (reading A16, A17)


# ------------------------------------------------------------------------------------------
# test support: a second valid oracle (reading S4: any summation order of a Galerkin entry)
# ------------------------------------------------------------------------------------------
def test_set_level_values_refreshes_the_l1_diagonal_and_the_lu_and_nothing_else():
    """orc_set_level_values carries no arithmetic of the method: writing the stored values back changes no bit of a
    solve; writing other values changes exactly A_l, its l1 diagonal (S8: numpy row sums) and, on the coarsest level,
    the direct solve (numpy.linalg.solve on the new dense matrix).  resum_galerkin_two_stage then yields a hierarchy
    whose operators are scipy's P^T (A P) to rounding: a second valid oracle, a little apart from the first."""
    from tests.reference_global import resum_galerkin_two_stage
    p = wl.make_config(5, 64)
    a, b, c = make_oracle(p), make_oracle(p), make_oracle(p)
    L = a.num_levels - 1
    assert L >= 2
    for l in range(1, L + 1):                                   # the identity: same values back
        c.set_level_values(l, c.matrix(l, "A")[2])
    with pytest.raises(RuntimeError):
        c.set_level_values(0, c.matrix(0, "A")[2])              # A_0 is the problem statement, not replaceable
    moved = resum_galerkin_two_stage(b)
    assert len(moved) == L and 0.0 < max(moved) < 1e-12
    rng = np.random.default_rng(5)
    for l in range(1, L + 1):
        A_new = b.scipy_matrix(l, "A")
        assert not np.array_equal(A_new.data, a.matrix(l, "A")[2]) or moved[l - 1] == 0.0
        assert np.allclose(b.dinv(l), l1_dinv(A_new), rtol=1e-14, atol=0)          # refreshed from the NEW values
        if moved[l - 1] > 1e-15:
            assert not np.allclose(b.dinv(l), a.dinv(l), rtol=1e-17, atol=0)
        # the product it was built from, recomputed here from the getters
        ref = (b.scipy_matrix(l - 1, "P").T @ (b.scipy_matrix(l - 1, "A") @ b.scipy_matrix(l - 1, "P"))).toarray()
        assert np.abs(A_new.toarray() - ref).max() == 0.0
        # P_l and the C/F splitting are untouched
        if l < L:
            assert np.array_equal(b.matrix(l, "P")[2], a.matrix(l, "P")[2]) and np.array_equal(b.cf(l), a.cf(l))
    rhs = rng.uniform(-1, 1, b.level_size(L)[0])
    want = np.linalg.solve(b.scipy_matrix(L, "A").toarray(), rhs)
    assert np.abs(b.coarse_solve(rhs) - want).max() <= 1e-9 * np.abs(want).max()
    xa, xb, xc = np.zeros(p.n), np.zeros(p.n), np.zeros(p.n)
    ra = a.solve(p.b, xa, 3, 2, 1)
    rb = b.solve(p.b, xb, 3, 2, 1)
    rc = c.solve(p.b, xc, 3, 2, 1)
    assert np.array_equal(xa, xc) and np.array_equal(ra, rc)
    d = np.abs(xa - xb).max() / np.abs(xa).max()
    assert 0.0 < d < 1e-8 and np.allclose(ra, rb, rtol=1e-7)
