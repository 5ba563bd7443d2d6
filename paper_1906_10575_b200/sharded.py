"""Exchange driver of the sharded AMG-DD cycle (include/amgdd.h, "sharding over ranks"; paper section 5, Alg. 5).

The library packs and unpacks on the device; THIS module only moves the packed buffers between the ranks
(plumbing: torch.distributed, or plain copies between ranks that live in one process) and runs the index protocol of
the redundancy removal once after setup.  No arithmetic of the method happens here.

Two communicators with the same interface:
  LocalComm(R)  all R ranks live in this process (tests on one GPU or on the CPU: handles / plans of every rank)
  DistComm()    one rank per process, torch.distributed initialised by the caller (nccl on GPUs, gloo for the protocol)
Every driver function takes dicts keyed by the ranks that live in this process.
"""
from __future__ import annotations

import numpy as np

from . import (amgdd_get_shard_plan, amgdd_shard_commit, amgdd_shard_local_solve, amgdd_shard_owned_count,
               amgdd_shard_pack_owned, amgdd_shard_plan_apply_drop, amgdd_shard_plan_info, amgdd_shard_plan_list,
               amgdd_shard_plan_recv_filter, amgdd_shard_sqnorm, amgdd_shard_stage_counts, amgdd_shard_stage_pack,
               amgdd_shard_stage_unpack, amgdd_shard_unpack_owned, amgdd_solve)


class LocalComm:
    """All ranks in one process."""

    def __init__(self, nranks):
        self.nranks = nranks
        self.local_ranks = list(range(nranks))

    def exchange_objects(self, outgoing):
        """outgoing[src][dst] -> incoming[dst][src]"""
        return {d: {s: outgoing[s][d] for s in self.local_ranks} for d in self.local_ranks}

    def exchange_values(self, sendbufs, send_counts, recv_counts):
        """sendbufs[src]: tensor, rank after rank as send_counts[src] says -> recvbufs[dst] likewise by recv_counts[dst]"""
        import torch
        out = {}
        for d in self.local_ranks:
            parts = []
            for s in self.local_ranks:
                off = int(send_counts[s][:d].sum())
                parts.append(sendbufs[s][off:off + int(send_counts[s][d])])
            out[d] = torch.cat(parts) if parts else sendbufs[d][:0]
            assert out[d].numel() == int(recv_counts[d].sum())
        return out

    def allgather_values(self, bufs):
        """bufs[src] -> {dst: [buf of rank 0, buf of rank 1, ...]}"""
        return {d: [bufs[s] for s in self.local_ranks] for d in self.local_ranks}

    def allreduce_sum(self, vals):
        tot = sum(vals[r] for r in self.local_ranks)
        return {r: tot for r in self.local_ranks}


class DistComm:
    """One rank per process over torch.distributed (initialised by the caller)."""

    def __init__(self):
        import torch.distributed as dist
        self.dist = dist
        self.nranks = dist.get_world_size()
        self.rank = dist.get_rank()
        self.local_ranks = [self.rank]

    def exchange_objects(self, outgoing):
        gathered = [None] * self.nranks
        self.dist.all_gather_object(gathered, outgoing[self.rank])           # setup only: simple, backend-agnostic
        return {self.rank: {s: gathered[s][self.rank] for s in range(self.nranks)}}

    def exchange_values(self, sendbufs, send_counts, recv_counts):
        import torch
        r = self.rank
        recv = torch.empty(int(recv_counts[r].sum()), dtype=torch.float64, device=sendbufs[r].device)
        self.dist.all_to_all_single(recv, sendbufs[r], [int(c) for c in recv_counts[r]], [int(c) for c in send_counts[r]])
        return {r: recv}

    def allgather_values(self, bufs, counts=None):
        import torch
        r = self.rank
        outs = [torch.empty(int(c), dtype=torch.float64, device=bufs[r].device) for c in counts]
        self.dist.all_gather(outs, bufs[r])
        return {r: outs}

    def allreduce_sum(self, vals):
        import torch
        t = torch.tensor([vals[self.rank]], dtype=torch.float64)
        if self.dist.get_backend() == "nccl":
            t = t.cuda()
        self.dist.all_reduce(t)
        return {self.rank: float(t.item())}


def run_index_protocol(plans, comm):
    """The announcement / redundancy-removal rounds of include/amgdd.h over every stage.  plans: {rank: ShardPlan}."""
    info = {r: amgdd_shard_plan_info(p) for r, p in plans.items()}
    nstages = next(iter(info.values()))["num_stages"]
    R = comm.nranks
    for stage in range(nstages):
        announced = comm.exchange_objects({r: {d: amgdd_shard_plan_list(plans[r], 0, stage, d) for d in range(R)} for r in plans})
        redundant = {}
        for d in plans:                                                    # receivers: sources in ascending rank
            redundant[d] = {s: amgdd_shard_plan_recv_filter(plans[d], stage, s, announced[d][s]) for s in range(R)}
        back = comm.exchange_objects(redundant)
        for s in plans:
            for d in range(R):
                amgdd_shard_plan_apply_drop(plans[s], stage, d, back[s][d])


def setup_exchange(handles, comm):
    """After amgdd_setup_shard on every rank: index protocol, then upload of the final lists."""
    plans = {r: amgdd_get_shard_plan(h) for r, h in handles.items()}
    run_index_protocol(plans, comm)
    for h in handles.values():
        amgdd_shard_commit(h)
        h._stage_cache = {}            # counts and send buffers per stage live ON the handle object and die with it
    return plans


def _same_stream(h, tensor):
    """The library enqueues pack / unpack / solve on the handle's stream; the exchange (torch.distributed, torch.cat, the
    buffers) runs on torch's current stream.  Nothing orders the two, so they must be the same stream."""
    import torch
    mine = int(getattr(h, "_stream", 0) or 0)
    cur = int(torch.cuda.current_stream(tensor.device).cuda_stream) if tensor.is_cuda else 0
    if mine != cur:
        raise RuntimeError(f"the handle works on CUDA stream {mine:#x} but torch's current stream is {cur:#x}: the packed buffers would "
                           "race with the exchange; call amgdd_set_stream(h) under the stream the cycle runs on")


def sharded_cycle(handles, b, x, comm, num_fac_cycles=2, relax_sweeps=1, want_norm=False):
    """One AMG-DD cycle with the Alg. 5 exchange.  handles, b, x: {rank: ...} for the ranks of this process (x in/out:
    valid on the rank's dofs).  Returns ||b - A x||_2 of the iterate the cycle STARTED from if want_norm."""
    import torch
    R = comm.nranks
    for r, h in handles.items():
        _same_stream(h, x[r])
        if not hasattr(h, "_stage_cache"):
            h._stage_cache = {}
    h0 = next(iter(handles.values()))
    if "nstages" not in h0._stage_cache:
        h0._stage_cache["nstages"] = 2 * (amgdd_shard_plan_info(amgdd_get_shard_plan(h0))["num_levels"] - 1) + 2
    nstages = h0._stage_cache["nstages"]
    norm = None
    for stage in range(nstages):
        sc, rc, bufs = {}, {}, {}
        for r, h in handles.items():
            if stage not in h._stage_cache:                                # counts and the send buffer of a stage never change
                s_cnt, r_cnt = amgdd_shard_stage_counts(h, stage, R)
                h._stage_cache[stage] = (s_cnt, r_cnt, torch.empty(int(s_cnt.sum()), dtype=torch.float64, device=x[r].device))
            sc[r], rc[r], bufs[r] = h._stage_cache[stage]
            amgdd_shard_stage_pack(h, stage, b[r], x[r], bufs[r])
        if want_norm and stage == 1:                                       # the owned rows' r_0 was just computed
            sq = comm.allreduce_sum({r: amgdd_shard_sqnorm(h) for r, h in handles.items()})
            norm = float(np.sqrt(next(iter(sq.values()))))
        recv = comm.exchange_values(bufs, sc, rc)
        for r, h in handles.items():
            amgdd_shard_stage_unpack(h, stage, x[r], recv[r])
    for r, h in handles.items():
        amgdd_shard_local_solve(h, x[r], num_fac_cycles, relax_sweeps)
    return norm


def allgather_cycle(handles, b, x, comm, num_fac_cycles=2, relax_sweeps=1):
    """The simple alternative: all-gather x, then the unsharded global part redundantly on every
    rank and AlgFAC on the rank's subdomains (amgdd_solve on the shard handle)."""
    import torch
    R = comm.nranks
    bufs, counts = {}, None
    for r, h in handles.items():
        _same_stream(h, x[r])
        counts = [amgdd_shard_owned_count(h, q) for q in range(R)]
        bufs[r] = torch.empty(counts[r], dtype=torch.float64, device=x[r].device)
        amgdd_shard_pack_owned(h, x[r], bufs[r])
    gathered = comm.allgather_values(bufs, counts) if isinstance(comm, DistComm) else comm.allgather_values(bufs)
    norms = {}
    for r, h in handles.items():
        for q in range(R):
            if q != r:
                amgdd_shard_unpack_owned(h, q, gathered[r][q], x[r])
        norms[r] = float(amgdd_solve(h, b[r], x[r], 1, num_fac_cycles, relax_sweeps)[0])     # ||b - A x|| of the gathered iterate
    return norms
