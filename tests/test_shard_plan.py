"""NEXT 4: the index sets of the sharded cycle -- rank ownership on every level, the mat-vec
halos of Alg. 2 and the Psi / Psi_c sets of the residual communication algorithm (paper section 5; Alg. 5)
with the redundancy removal of P:250 -- against a brute-force restatement written here from the ORACLE's hierarchy and
composite grids (independent code): who owns each point, which points of whose composite grid a rank needs, graph
distances by all-pairs shortest paths.  No GPU: amgdd_shard_plan_create rebuilds the hierarchy on the host."""
import numpy as np
import pytest
import scipy.sparse as sp
from scipy.sparse.csgraph import shortest_path

import workloads as wl
from oracle import Oracle


def build_plans(p, R):
    import paper_1906_10575_b200 as m
    return {r: m.amgdd_shard_plan_create(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.max_levels, p.theta,
                                         p.coarse_max, rank=r, nranks=R) for r in range(R)}


def oracle_of(p):
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, p.theta, p.max_levels, p.coarse_max)
    o.set_partition(p.num_subdomains, p.owner, p.eta, p.num_ghost)
    return o


def brute_owner_rank(o, p, R):
    """Omega_l^r: level 0 from the owner array (rank of subdomain q = floor(q R / P)); level l + 1: coarse images of the C-points
    (coarse index = rank among the C-points, S2)."""
    own = [(p.owner.astype(np.int64) * R // p.num_subdomains).astype(np.int32)]
    for l in range(o.num_levels - 1):
        own.append(own[l][o.cf(l) > 0])
    return own


def check_everything(p, R, plans):
    import paper_1906_10575_b200 as m
    from paper_1906_10575_b200.sharded import LocalComm, run_index_protocol
    o = oracle_of(p)
    L = o.num_levels - 1
    info = m.amgdd_shard_plan_info(plans[0])
    assert info["num_levels"] == L + 1 and info["num_stages"] == 2 * L + 2 and info["nranks"] == R
    own = brute_owner_rank(o, p, R)
    roff = [m.amgdd_shard_plan_level(plans[0], l)[1] for l in range(L + 1)]
    for r in range(R):
        for l in range(L + 1):
            assert np.array_equal(m.amgdd_shard_plan_owner_rank(plans[r], l), own[l])
        assert m.amgdd_shard_plan_info(plans[r])["sub_lo"] == -(-r * p.num_subdomains // R)
    # ---- the raw Psi of every Alg. 5 stage is the set the paper defines (all-pairs shortest paths) ----
    A = [o.scipy_matrix(l, "A") for l in range(L + 1)]
    for l in range(L + 1):
        n_l = A[l].shape[0]
        if n_l > 1500:
            continue
        dist = shortest_path(sp.csr_matrix((np.ones(A[l].nnz), A[l].indices, A[l].indptr), shape=A[l].shape), unweighted=True)
        stage = L + 1 + (L - l)
        for r in range(R):
            mine = np.flatnonzero(own[l] == r)
            for q in range(R):
                if q == r:
                    continue
                theirs = np.flatnonzero(own[l] == q)
                if l == L:
                    psi = mine
                elif len(theirs) == 0 or len(mine) == 0:
                    psi = mine[:0]
                else:
                    psi = mine[dist[np.ix_(mine, theirs)].min(axis=1) <= p.eta]
                raw = m.amgdd_shard_plan_list(plans[r], 0, stage, q)
                at_l = raw[(raw >= roff[l]) & (raw < roff[l] + n_l)] - roff[l]
                assert np.array_equal(at_l, psi), (l, r, q)
                if len(psi) == 0:
                    assert len(raw) == 0                                   # not a neighbour: nothing at all is sent
    # ---- protocol, then a token simulation of the staged exchange ----
    run_index_protocol(plans, LocalComm(R))
    need = []                                                              # N_l^r = union of D_l^p over the rank's subdomains
    for r in range(R):
        lo, hi = -(-r * p.num_subdomains // R), -(-(r + 1) * p.num_subdomains // R)
        per_level = [np.zeros(A[l].shape[0], bool) for l in range(L + 1)]
        for q in range(lo, hi):
            for l in range(L + 1):
                per_level[l][o.composite(q, l)[0]] = True
        need.append(per_level)
    total = roff[L] + A[L].shape[0]
    valid_r = [np.zeros(total, bool) for _ in range(R)]
    for r in range(R):
        for l in range(L + 1):
            valid_r[r][roff[l] + np.flatnonzero(own[l] == r)] = True
    valid_x = [own[0] == r for r in range(R)]
    A0 = A[0].tocsr()
    for stage in range(2 * L + 2):
        vec = m.amgdd_shard_plan_stage_vector(plans[0], stage)
        valid = valid_x if vec == 0 else valid_r
        snap = [v.copy() for v in valid]                                   # what a rank holds when the stage starts
        for d in range(R):
            got = []
            for s in range(R):
                snd = m.amgdd_shard_plan_list(plans[s], 0, stage, d)
                rcv = m.amgdd_shard_plan_list(plans[d], 1, stage, s)
                assert np.array_equal(snd, rcv), "both sides must agree on the list and its order"
                assert s != d or len(snd) == 0
                assert snap[s][snd].all(), f"stage {stage}: rank {s} forwards a value it does not hold"
                assert not snap[d][snd].any(), f"stage {stage}: rank {d} receives a value it already holds"
                got.append(snd)
            got = np.concatenate(got) if got else np.zeros(0, np.int64)
            assert len(np.unique(got)) == len(got), "a position arrives twice in one stage"
            valid[d][got] = True
        if stage == 0:                                                     # x halo: exactly the columns of the owned rows of A_0
            for r in range(R):
                cols = np.unique(A0[np.flatnonzero(own[0] == r)].indices)
                assert valid_x[r][cols].all()
        elif stage <= L:                                                   # r_l halo: the columns of the owned rows of R_l = P_l^T
            l = stage - 1
            Rl = o.scipy_matrix(l, "P").T.tocsr()
            for r in range(R):
                cols = np.unique(Rl[np.flatnonzero(own[l + 1] == r)].indices)
                assert valid_r[r][roff[l] + cols].all()
    for r in range(R):
        for l in range(L + 1):
            idx = roff[l] + np.flatnonzero(need[r][l])
            assert valid_r[r][idx].all(), f"rank {r} misses residuals of its composite grid on level {l}"


@pytest.mark.parametrize("cfg,scale,R,kw", [(1, None, 2, {}), (1, 37, 3, {"parts_per_dim": 3}), (2, 16, 2, {"parts_per_dim": 2}),
                                             (4, 24, 4, {}), (5, 64, 2, {"parts_per_dim": 2}), (1, 21, 4, {"eta": 2, "parts_per_dim": 2})])
def test_shard_index_sets_against_brute_force(cfg, scale, R, kw):
    p = wl.make_config(cfg, scale, **kw)
    check_everything(p, R, build_plans(p, R))


def test_shard_degenerate_hierarchies():
    """L = 0 (the whole problem is the coarsest level: every rank sends all it owns to every other rank, reading A5) and
    eta = 0 (Psi = the points adjacent to nothing: only Psi_c structures and the halos move)."""
    import copy
    p = copy.copy(wl.make_config(1, 7, parts_per_dim=2))
    p.coarse_max = 64
    check_everything(p, 2, build_plans(p, 2))
    p = wl.make_config(2, 16, parts_per_dim=2, eta=0)
    o = oracle_of(p)
    x = np.zeros(p.n)
    o.cycle(p.b, x, 1, 1)
    if o.dropped() == 0:                                  # (with eta = 0 the composite grids may not be closed under interpolation, A7)
        check_everything(p, 2, build_plans(p, 2))


def test_one_rank_exchanges_nothing():
    import paper_1906_10575_b200 as m
    p = wl.make_config(1)
    plan = build_plans(p, 1)[0]
    for stage in range(m.amgdd_shard_plan_info(plan)["num_stages"]):
        assert len(m.amgdd_shard_plan_list(plan, 0, stage, 0)) == 0


def test_shard_argument_checks():
    import paper_1906_10575_b200 as m
    p = wl.make_config(1)
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_shard_plan_create(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, rank=2, nranks=2)
    assert e.value.code == -1
    with pytest.raises(m.AmgddError):
        m.amgdd_shard_plan_create(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, rank=0, nranks=5)   # more ranks than subdomains


def test_index_protocol_is_refused_a_second_time():
    """The redundancy removal marks positions as held for good, so a second pass would drop every send list.  The C ABI
    refuses it (AMGDD_ERR_BAD_ARG) and leaves the lists of the first pass as they are."""
    import paper_1906_10575_b200 as m
    from paper_1906_10575_b200.sharded import LocalComm, run_index_protocol
    p = wl.make_config(1, 21, parts_per_dim=2)
    R = 2
    plans = {r: m.amgdd_shard_plan_create(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.max_levels,
                                          p.theta, p.coarse_max, rank=r, nranks=R) for r in range(R)}
    run_index_protocol(plans, LocalComm(R))
    nstages = m.amgdd_shard_plan_info(plans[0])["num_stages"]
    before = {(r, w, s, q): m.amgdd_shard_plan_list(plans[r], w, s, q).copy()
              for r in range(R) for w in (0, 1) for s in range(nstages) for q in range(R)}
    assert sum(len(v) for v in before.values()) > 0
    with pytest.raises(m.AmgddError) as e:
        run_index_protocol(plans, LocalComm(R))
    assert e.value.code == -1 and "already" in str(e.value)
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_shard_plan_apply_drop(plans[0], 0, 1, before[(0, 0, 0, 1)])
    assert e.value.code == -1 and "already" in str(e.value)
    for key, want in before.items():
        r, w, s, q = key
        assert np.array_equal(m.amgdd_shard_plan_list(plans[r], w, s, q), want), key
