"""NEXT 4 on one GPU: R virtual ranks in one process (one shard handle per rank on the same device, the exchange of every
stage done by copies between their buffers).  The sharded cycle -- mat-vec halos, the Alg. 5 residual exchange with
forwarding, AlgFAC on the rank's subdomains -- must leave x BIT-IDENTICAL to the unsharded amgdd_solve (the same row
sums in the same order, only computed by the rank that owns the row), for the Alg. 5 exchange and for the all-gather
alternative.  Before each cycle a rank's x is poisoned with NaN outside its own dofs, and three cycles are compared, so a
halo value that was not exchanged, or a residual left over from the cycle before, cannot go unnoticed."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


def _setup(p, R):
    import torch
    import paper_1906_10575_b200 as m
    from paper_1906_10575_b200.sharded import LocalComm, setup_exchange
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    handles = {r: m.amgdd_setup_shard(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.num_ghost, p.max_levels,
                                      p.theta, p.coarse_max, rank=r, nranks=R) for r in range(R)}
    comm = LocalComm(R)
    plans = setup_exchange(handles, comm)
    return m, handles, comm, plans


@pytest.mark.parametrize("cfg,scale,R,kw", [(1, None, 2, {}), (2, 32, 2, {}), (4, 48, 4, {}), (4, 48, 3, {}), (5, 256, 4, {}),
                                             (3, 32, 2, {"eta": 2})])
def test_sharded_cycle_is_bit_identical(cfg, scale, R, kw):
    import torch
    from paper_1906_10575_b200.sharded import allgather_cycle, sharded_cycle
    p = wl.make_config(cfg, scale, **kw)
    m, handles, comm, plans = _setup(p, R)
    own0 = torch.from_numpy(m.amgdd_shard_plan_owner_rank(plans[0], 0)).cuda()
    href = m.amgdd_setup(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.num_ghost, p.max_levels, p.theta, p.coarse_max)
    b = torch.from_numpy(p.b).cuda()
    xref = torch.zeros(p.n, dtype=torch.float64, device="cuda")
    ncyc = 3
    ref = m.amgdd_solve(href, b, xref.clone(), 0)          # ||b||
    for mode in ("alg5", "allgather"):
        xr = torch.zeros(p.n, dtype=torch.float64, device="cuda")
        # every rank starts from the same x = 0; afterwards a rank's x is valid on its own dofs only
        x = {r: torch.zeros(p.n, dtype=torch.float64, device="cuda") for r in range(R)}
        bb = {r: b for r in range(R)}
        for k in range(ncyc):
            res = m.amgdd_solve(href, b, xr, 1, p.num_fac_cycles, p.relax_sweeps)
            if mode == "alg5":
                for r in range(R):                         # poison what the rank does not own
                    x[r][own0 != r] = float("nan")
                norm = sharded_cycle(handles, bb, x, comm, p.num_fac_cycles, p.relax_sweeps, want_norm=True)
            else:
                norm = allgather_cycle(handles, bb, x, comm, p.num_fac_cycles, p.relax_sweeps)[0]
            assert abs(norm - res[0]) <= 1e-13 * res[0], (mode, k, norm, res[0])
            # assemble x from the ranks' own dofs
            xs = torch.zeros_like(xr)
            for r in range(R):
                xs[own0 == r] = x[r][own0 == r]
            assert torch.equal(xs, xr), f"{mode}: x differs from the unsharded solve after cycle {k + 1}"
    assert ref[0] > 0
    for h in handles.values():
        m.amgdd_destroy(h)
    m.amgdd_destroy(href)


def test_sharded_cycle_with_the_cf_smoother_and_two_sweeps():
    import torch
    from paper_1906_10575_b200.sharded import sharded_cycle
    p = wl.make_config(2, 32)
    R = 4
    m, handles, comm, plans = _setup(p, R)
    own0 = torch.from_numpy(m.amgdd_shard_plan_owner_rank(plans[0], 0)).cuda()
    href = m.amgdd_setup(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.num_ghost, p.max_levels, p.theta, p.coarse_max)
    for h in list(handles.values()) + [href]:
        m.amgdd_set_smoother(h, 1)
    b = torch.from_numpy(p.b).cuda()
    xr = torch.zeros(p.n, dtype=torch.float64, device="cuda")
    x = {r: torch.zeros(p.n, dtype=torch.float64, device="cuda") for r in range(R)}
    for k in range(2):
        m.amgdd_solve(href, b, xr, 1, 3, 2)
        sharded_cycle(handles, {r: b for r in range(R)}, x, comm, 3, 2)
        xs = torch.zeros_like(xr)
        for r in range(R):
            xs[own0 == r] = x[r][own0 == r]
        assert torch.equal(xs, xr)


def test_shard_handle_reports_local_subdomains():
    import paper_1906_10575_b200 as m
    p = wl.make_config(2, 32)
    R = 3
    _, handles, _, plans = _setup(p, R)
    tot = 0
    for r in range(R):
        info = m.amgdd_shard_plan_info(plans[r])
        st = m.amgdd_get_stats(handles[r])
        assert st["num_subdomains"] == info["sub_hi"] - info["sub_lo"]
        tot += st["num_subdomains"]
    assert tot == p.num_subdomains


def test_sharded_cycle_refuses_a_handle_on_another_stream():
    """The exchange runs on torch's current stream, the library on the handle's: the driver checks that they are one."""
    import torch
    from paper_1906_10575_b200.sharded import allgather_cycle, sharded_cycle
    p = wl.make_config(1)
    m, handles, comm, plans = _setup(p, 2)
    b = torch.from_numpy(p.b).cuda()
    x = {r: torch.zeros(p.n, dtype=torch.float64, device="cuda") for r in range(2)}
    bb = {r: b for r in range(2)}
    side = torch.cuda.Stream()
    m.amgdd_set_stream(handles[1], side)
    for cycle in (sharded_cycle, allgather_cycle):
        with pytest.raises(RuntimeError, match="current stream"):
            cycle(handles, bb, x, comm, p.num_fac_cycles, p.relax_sweeps)
    with torch.cuda.stream(side):                      # under that stream for both handles: accepted
        m.amgdd_set_stream(handles[0], side)
        sharded_cycle(handles, bb, x, comm, p.num_fac_cycles, p.relax_sweeps)
    side.synchronize()
    assert hasattr(handles[0], "_stage_cache") and "nstages" in handles[0]._stage_cache
    for h in handles.values():
        m.amgdd_destroy(h)


@pytest.mark.parametrize("cfg,scale,R", [(4, 24, 2), (2, 32, 3)])
def test_sharded_cycle_against_the_oracle(cfg, scale, R):
    """The sharded cycle (Alg. 5 exchange) compared with the ORACLE directly, not through the unsharded library
    path: residual norms and the x assembled from the ranks' own dofs, per cycle, at the plain 1e-10 bar."""
    import torch
    from oracle import Oracle, max_threads
    from paper_1906_10575_b200.sharded import sharded_cycle
    p = wl.make_config(cfg, scale)
    m, handles, comm, plans = _setup(p, R)
    own0 = torch.from_numpy(m.amgdd_shard_plan_owner_rank(plans[0], 0)).cuda()
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, p.theta, p.max_levels, p.coarse_max)
    o.set_partition(p.num_subdomains, p.owner, p.eta, p.num_ghost)
    b = torch.from_numpy(p.b).cuda()
    x = {r: torch.zeros(p.n, dtype=torch.float64, device="cuda") for r in range(R)}
    bb = {r: b for r in range(R)}
    xo = np.zeros(p.n)
    for k in range(3):
        r_before = o.residual_norm(p.b, xo)
        for r in range(R):
            x[r][own0 != r] = float("nan")
        norm = sharded_cycle(handles, bb, x, comm, p.num_fac_cycles, p.relax_sweeps, want_norm=True)
        o.cycle(p.b, xo, p.num_fac_cycles, p.relax_sweeps, nthreads=max_threads())
        assert abs(norm - r_before) <= 1e-10 * r_before, (k, norm, r_before)
        xs = torch.zeros(p.n, dtype=torch.float64, device="cuda")
        for r in range(R):
            xs[own0 == r] = x[r][own0 == r]
        err = np.abs(xs.cpu().numpy() - xo).max()
        assert err <= 1e-10 * np.abs(xo).max(), (k, err)
    for h in handles.values():
        m.amgdd_destroy(h)
