"""NEXT 4: the index protocol of the sharded cycle (announcement, redundancy removal of P:250) run by TWO processes over
torch.distributed with the gloo backend (CPU): every rank builds only its own plan, the lists travel through the
communicator, and the result must equal the in-process run that tests/test_shard_plan.py checks against brute force."""
import os
import socket

import numpy as np
import pytest


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, cfg, scale, kw, out_dir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import workloads as wl
    import paper_1906_10575_b200 as m
    from paper_1906_10575_b200.sharded import DistComm, run_index_protocol
    p = wl.make_config(cfg, scale, **kw)
    plan = m.amgdd_shard_plan_create(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.max_levels, p.theta,
                                     p.coarse_max, rank=rank, nranks=world)
    run_index_protocol({rank: plan}, DistComm())
    nst = m.amgdd_shard_plan_info(plan)["num_stages"]
    lists = {(w, st, q): m.amgdd_shard_plan_list(plan, w, st, q) for w in (0, 1) for st in range(nst) for q in range(world)}
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), **{f"{w}_{st}_{q}": v for (w, st, q), v in lists.items()})
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("cfg,scale,kw", [(1, None, {}), (4, 24, {})])
def test_index_protocol_over_gloo_world_size_2(cfg, scale, kw, tmp_path):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), cfg, scale, kw, str(tmp_path)), nprocs=world, join=True)
    import workloads as wl
    import paper_1906_10575_b200 as m
    from paper_1906_10575_b200.sharded import LocalComm, run_index_protocol
    from tests.test_shard_plan import build_plans
    p = wl.make_config(cfg, scale, **kw)
    plans = build_plans(p, world)
    run_index_protocol(plans, LocalComm(world))
    nst = m.amgdd_shard_plan_info(plans[0])["num_stages"]
    moved = 0
    for r in range(world):
        got = np.load(os.path.join(str(tmp_path), f"rank{r}.npz"))
        for w in (0, 1):
            for st in range(nst):
                for q in range(world):
                    ref = m.amgdd_shard_plan_list(plans[r], w, st, q)
                    assert np.array_equal(got[f"{w}_{st}_{q}"], ref), (r, w, st, q)
                    moved += len(ref)
    assert moved > 0
