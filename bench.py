#!/usr/bin/env python
"""bench.py -- AMG-DD cycle time on B200 (metric of BASELINE.json: "AMG-DD cycle time (ms),
FAC-sweep HBM GB/s vs peak, residual drop/cycle").

A "step" is ONE AMG-DD cycle (Alg. 2) over the whole workload: global residual and
its norm (a1, a11), restriction to all levels (a2), and the persistent AlgFAC kernel that gathers
the residuals, runs num_fac_cycles V(1,1) AlgFAC cycles on every subdomain and updates the owned
dofs (a3-a10).  Default workload: BASELINE.json configs[3] (3D variable-coefficient diffusion,
192^3, 4096 subdomains, eta = 2), the largest config that fits one B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config {1,2,3,4,5}] [--scale S] [--impl reference]

One JSON line on stdout (rank 0).  With --impl reference the CPU oracle is timed instead (on a
bounded sample of the same workload); see DESIGN.md section 13 (Measurement).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "amgdd_cycle_time"
UNIT = "ms"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--scale", type=int, default=None, help="grid edge override (smaller instance of the recipe)")
    ap.add_argument("--eta", type=int, default=None)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-sample", type=int, default=None, help="subdomains in the oracle's timed sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the short runs of configs 1, 2, 5 after the default config-4 line")
    ap.add_argument("--all-configs", action="store_true", help="per_config also runs config 3 at eta = 1 (112 GB on the device, long setup)")
    ap.add_argument("--smoother", type=int, default=0, choices=[0, 1], help="0: l1-Jacobi (BASELINE), 1: CF l1-Jacobi (P:275)")
    ap.add_argument("--shard", default=None, choices=["alg5", "allgather"],
                    help="under torchrun: shard the subdomains over the ranks (NEXT 4; Alg. 5 exchange or all-gather of x) "
                         "instead of running replicas; unmeasured on multi-GPU hardware (DESIGN.md section 8)")
    return ap.parse_args()


def workload_name(p, args):
    return f"{p.name}-P{p.num_subdomains}-eta{p.eta}-fac{p.num_fac_cycles}xV({p.relax_sweeps},{p.relax_sweeps})" + ("-cfjacobi" if args.smoother else "")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""

    QUERY = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 6:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for nm, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def kernel_source_hash():
    """Identifies the AlgFAC kernel a committed ncu capture belongs to: sha256 over the kernel and the stream layout."""
    import hashlib
    hsh = hashlib.sha256()
    for name in ("amgdd_fac.cu", "amgdd_stream.hpp"):
        with open(os.path.join(ROOT, "paper_1906_10575_b200", "csrc", name), "rb") as f:
            hsh.update(f.read())
    return hsh.hexdigest()[:16]


def ncu_traffic(workload):
    """DRAM bytes per AlgFAC launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed
    `ncu --set full` capture of this workload -- only if that capture was taken with the kernel source that is
    running now (profiles/fac_kernel_traffic.json records the hash); otherwise None."""
    path = os.path.join(ROOT, "profiles", "fac_kernel_traffic.json")
    try:
        d = json.load(open(path))
        if d.get("source_hash") != kernel_source_hash():
            return None
        return d.get("workloads", {}).get(workload)
    except Exception:
        return None


# ---------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline of the b200 arm, and the whole --impl reference arm)
# ---------------------------------------------------------------------------------------------
def oracle_time_per_cycle(p, sample, steps, warmup, smoother=0, sample_1thread=None):
    """Times the oracle AS IT STANDS on a bounded sample: every step runs Alg. 2's global residual +
    restriction over the whole problem and AlgFAC on `sample` subdomains (spread evenly over the
    partition).  Timed with all host cores (one OpenMP thread per core, `value`) and, on a smaller sample, with ONE
    thread (`value_1thread`)."""
    from oracle import Oracle, max_threads
    t0 = time.time()
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, p.theta, p.max_levels, p.coarse_max)
    o.set_partition(p.num_subdomains, p.owner, p.eta, p.num_ghost)
    o.set_smoother(smoother)
    setup_s = time.time() - t0
    nthreads = max_threads()
    sample = max(1, min(sample, p.num_subdomains))
    subs = np.unique(np.linspace(0, p.num_subdomains - 1, sample).astype(np.int32))
    x = np.zeros(p.n)

    def timed(sub_list, nt):
        times = []
        for _ in range(steps):
            t = time.time()
            o.cycle(p.b, x, p.num_fac_cycles, p.relax_sweeps, subdomains=sub_list, nthreads=nt)
            times.append(time.time() - t)
        return times

    for _ in range(max(1, warmup)):
        o.cycle(p.b, x, p.num_fac_cycles, p.relax_sweeps, subdomains=subs, nthreads=nthreads)   # also builds the composite grids (setup)
    n1 = max(1, min(len(subs), sample_1thread or min(64, max(1, len(subs) // 4))))
    subs1 = subs[np.unique(np.linspace(0, len(subs) - 1, n1).astype(int))]
    one = subs[len(subs) // 2:len(subs) // 2 + 1]

    def per_cycle(sub_list, nt):
        """A step costs g + a * (subdomains in it): g = Alg. 2's global residual + restriction (run in full every step),
        a = AlgFAC per subdomain.  Two sample sizes give both; the cycle of the whole workload costs g + a * P."""
        t_s, t_1 = float(np.mean(timed(sub_list, nt))), float(np.mean(timed(one, nt)))
        if len(sub_list) > 1:
            a = max(0.0, (t_s - t_1) / (len(sub_list) - 1))
            g = max(0.0, t_1 - a)
        else:
            a, g = t_s, 0.0
        return 1e3 * (g + a * p.num_subdomains), t_s, g

    est_ms, t_all, g_all = per_cycle(subs, nthreads)
    est1_ms, t_one, g_one = per_cycle(subs1, 1)
    return {"value": est_ms, "unit": UNIT, "cores": nthreads, "kind": "oracle",
            "value_1thread": est1_ms,
            "sample": f"all cores: {len(subs)} of {p.num_subdomains} subdomains per step, {steps} timed steps after {max(1, warmup)} "
                      f"warm-up; one thread: {len(subs1)} subdomains per step, {steps} steps; every step also runs the global "
                      f"residual+restriction in full, so a second timing with ONE subdomain separates that part (g) from the cost "
                      f"per subdomain (a); per-cycle value = g + a x P; oracle setup {setup_s:.1f}s not timed",
            "sample_seconds_per_step": t_all, "sample_seconds_per_step_1thread": t_one,
            "global_part_seconds": g_all, "global_part_seconds_1thread": g_one,
            "steps_timed": steps, "subdomains_all_cores": int(len(subs)), "subdomains_1thread": int(len(subs1))}


def default_cpu_sample(p):
    # about 20-30 s of CPU work in total: ~0.06 core-seconds per config-4 subdomain-cycle on the box's 16 cores
    # (config 4: 256 subdomains x 4 steps on all cores ~ 4 s, 64 subdomains x 3 steps on one thread ~ 12 s)
    # config 4: ALL 4096 subdomains on all cores (3 timed cycles of about 4.3 s each after one warm-up cycle that also builds the
    # composite grids), so the all-cores value is a measured full cycle, not an extrapolation; the one-thread leg stays sampled
    return {1: 4, 2: 64, 3: 16, 4: 4096, 5: 1024}.get(int(p.name[3]), 32)


def run_reference(args, p, rank, world):
    if rank != 0:
        return
    steps, warmup = args.steps, args.warmup
    sample = args.cpu_sample or default_cpu_sample(p)
    steps_cpu = max(1, min(steps, 3))
    cb = oracle_time_per_cycle(p, sample, steps_cpu, max(1, min(warmup, 1)), args.smoother)
    line = {
        "impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": cb["value"], "higher_is_better": False,
        "scaling": "weak" if args.gpus > 1 else "none", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(p, args), "n_dofs": p.n, "nnz": p.nnz, "subdomains": p.num_subdomains, "eta": p.eta,
                   "theta": p.theta, "fac_cycles_per_step": p.num_fac_cycles, "relax_sweeps": p.relax_sweeps},
        "note": "CPU oracle as it stands (cpu_baseline.sample says which subdomains a step ran: all of them on config 4), timed steps capped at 3",
        "cpu_baseline": cb,
        "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# B200 arm
# ---------------------------------------------------------------------------------------------
def measure_config(m, torch, cfg, steps, warmup, eta=None):
    """Short run of another BASELINE.json config for the `per_config` record (north_star: "report throughput on synthetic
    Poisson and variable-coefficient diffusion systems"): the same step as the headline line -- one AMG-DD cycle, asynchronous
    calls timed with CUDA events on the handle's stream -- plus the AlgFAC launch time from the library's own events."""
    import workloads as wl
    p = wl.make_config(cfg, None, eta=eta)
    t0 = time.time()
    h = m.amgdd_setup(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.num_ghost,
                      p.max_levels, p.theta, p.coarse_max)
    setup_s = time.time() - t0
    st = m.amgdd_get_stats(h)
    stream = torch.cuda.current_stream()
    m.amgdd_set_stream(h, stream)
    b = torch.from_numpy(p.b).cuda()
    x = torch.zeros(p.n, dtype=torch.float64, device="cuda")
    nfac, nu = p.num_fac_cycles, p.relax_sweeps
    res = m.amgdd_solve(h, b, x, min(p.num_cycles, 5), nfac, nu)
    x.zero_()
    for _ in range(max(3, warmup)):
        m.amgdd_solve(h, b, x, 1, nfac, nu, want_norms=False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(steps):
        m.amgdd_solve(h, b, x, 1, nfac, nu, want_norms=False)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_step = e0.elapsed_time(e1) / steps
    fac_ms = []
    for _ in range(steps):
        m.amgdd_solve(h, b, x, 1, nfac, nu)
        fac_ms.append(m.amgdd_last_solve_profile(h)["ms_fac"])
    fac = float(np.mean(fac_ms))
    peak, _ = measured_peak()
    model_bytes = st["model_bytes_fac_iter"][0] + (nfac - 1) * st["model_bytes_fac_iter"][1]
    stream_bytes = st["stream_bytes_fac_iter"][0] + (nfac - 1) * st["stream_bytes_fac_iter"][1]
    out = {"ms_per_step": ms_step, "fac_ms": fac, "frac": model_bytes / (fac * 1e-3) / 1e9 / peak,
           "frac_stream": stream_bytes / (fac * 1e-3) / 1e9 / peak, "stream_bytes_per_step": stream_bytes,
           "l2": "inputs larger than L2" if stream_bytes > 2 * 126e6 else "matrix streams fit the 126 MB L2: an L2-resident number, no flush between steps",
           "n_dofs": p.n, "subdomains": p.num_subdomains, "eta": p.eta, "levels": st["num_levels"], "device_bytes": st["device_bytes"],
           "setup_seconds": setup_s, "steps": steps, "residual_drop_per_cycle": (res[1:] / res[:-1]).tolist()[:3]}
    m.amgdd_destroy(h)
    del b, x
    torch.cuda.empty_cache()
    return p.name, out


def run_b200(args, p, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import paper_1906_10575_b200 as m

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the B200 arm has no CPU fallback")
    torch.cuda.set_device(local_rank)
    distributed = world > 1
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    if args.shard:
        return run_sharded(args, p, rank, world, local_rank, m, torch, dist)
    t0 = time.time()
    h = m.amgdd_setup(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.num_ghost,
                      p.max_levels, p.theta, p.coarse_max)
    setup_s = time.time() - t0
    st = m.amgdd_get_stats(h)
    m.amgdd_set_smoother(h, args.smoother)
    stream = torch.cuda.current_stream()
    m.amgdd_set_stream(h, stream)
    b = torch.from_numpy(p.b).cuda()
    x = torch.zeros(p.n, dtype=torch.float64, device="cuda")
    nfac, nu = p.num_fac_cycles, p.relax_sweeps

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- residual drop per cycle (also warms everything up) ----
    res = m.amgdd_solve(h, b, x, p.num_cycles, nfac, nu)
    drops = (res[1:] / res[:-1]).tolist()
    x.zero_()
    for _ in range(args.warmup):
        m.amgdd_solve(h, b, x, 1, nfac, nu, want_norms=False)

    # ---- timed region: exactly K steps, device-resident inputs ----
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        m.amgdd_solve(h, b, x, 1, nfac, nu, want_norms=False)
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)

    # ---- the dominant kernel: per-launch duration from the library's CUDA events on its stream ----
    x.zero_()
    if os.environ.get("AMGDD_FAC_PROFILE", "0") == "1":
        m.amgdd_debug_fac_op_cycles(h)                                   # clears the per-step counters
    fac_ms, launches = [], None
    for _ in range(args.steps):
        m.amgdd_solve(h, b, x, 1, nfac, nu)
        prof = m.amgdd_last_solve_profile(h)
        fac_ms.append(prof["ms_fac"])
        launches = prof["launches"]
    clocks = sampler.stop()
    fac_avg_ms = float(np.mean(fac_ms))
    fac_ops = m.amgdd_debug_fac_op_cycles(h) if os.environ.get("AMGDD_FAC_PROFILE", "0") == "1" else None   # exactly these cycles

    # ---- context: the paper's comparison method, one AMG V(1,1)-cycle on the same hierarchy (Alg. 1; Fig. 14-15) ----
    xv = torch.zeros(p.n, dtype=torch.float64, device="cuda")
    res_v = m.amgdd_vcycle(h, b, xv, p.num_cycles, 1, 1)
    for _ in range(2):
        m.amgdd_vcycle(h, b, xv, 1, 1, 1, want_norms=False)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        m.amgdd_vcycle(h, b, xv, 1, 1, 1, want_norms=False)
    e1.record(stream)
    barrier()
    vcycle_ms = e0.elapsed_time(e1) / args.steps
    del xv

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    bh = torch.from_numpy(p.b).pin_memory()
    xh = torch.zeros(p.n, dtype=torch.float64).pin_memory()
    for _ in range(2):
        m.amgdd_solve_host(h, bh, xh, 1, nfac, nu)
    barrier()
    t = time.perf_counter()
    for _ in range(args.steps):
        m.amgdd_solve_host(h, bh, xh, 1, nfac, nu)
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t) / args.steps

    ms_step = ms_total / args.steps
    vals = torch.tensor([ms_step, e2e_ms, fac_avg_ms], dtype=torch.float64, device="cuda")
    if distributed:
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)
    ms_step, e2e_ms, fac_avg_ms = [float(v) for v in vals.tolist()]

    if rank == 0:
        peak, peak_src = measured_peak()
        model_bytes = st["model_bytes_fac_iter"][0] + (nfac - 1) * st["model_bytes_fac_iter"][1]
        stream_bytes = st["stream_bytes_fac_iter"][0] + (nfac - 1) * st["stream_bytes_fac_iter"][1]
        useful_bytes = st["useful_bytes_fac_iter"][0] + (nfac - 1) * st["useful_bytes_fac_iter"][1]
        achieved = model_bytes / (fac_avg_ms * 1e-3) / 1e9
        wname = workload_name(p, args)
        traffic = ncu_traffic(wname)
        line = {
            "metric": METRIC, "value": ms_step, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": False,
            "scaling": "weak" if args.gpus > 1 else "none", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {
                "workload": wname, "n_dofs": p.n, "nnz": p.nnz, "subdomains": p.num_subdomains, "eta": p.eta,
                "theta": p.theta, "levels": st["num_levels"], "fac_cycles_per_step": nfac, "relax_sweeps": nu,
                "composite_overhead": st["overhead"], "device_bytes": st["device_bytes"],
                "l2_policy": "inputs larger than L2 (matrix streams %.1f GB per step)" % (stream_bytes / 1e9),
                "multi_gpu": "replicas only (north_star: one GPU, no sharding, no collectives)" if args.gpus > 1 else "single GPU",
                "setup_seconds": setup_s, "setup_seconds_hierarchy": st["setup_seconds_hierarchy"],
                "setup_seconds_composite": st["setup_seconds_composite"],
                "composite_assembly": "device" if st["assembled_on_device"] else "host",
            },
            "clocks": clocks,
            "e2e": {"value": e2e_ms, "unit": UNIT, "h2d_bytes_per_step": 2 * 8 * p.n, "d2h_bytes_per_step": 8 * p.n + 16},
            "gpu_launches": int(sum(launches)) * args.steps if launches else 0,
            "launches_per_step": launches,
            "residual_drop_per_cycle": drops,
            "residual_norms": res.tolist(),
            "phase_ms_per_step": {"fac_kernel": fac_avg_ms},
            "amg_vcycle_context": {
                "what": "one AMG V(1,1)-cycle (Alg. 1) on the same hierarchy and smoother, whole-level kernels, this GPU",
                "ms_per_cycle": vcycle_ms, "residual_drop_per_cycle": (res_v[1:] / res_v[:-1]).tolist(),
                "speedup_S_of_amgdd_over_amg": vcycle_ms / ms_step,
                "amgdd_asymptotic_factor_rho": float(np.prod(drops[-3:]) ** (1.0 / 3.0)),
                "effective_factor_rho_pow_S": float((np.prod(drops[-3:]) ** (1.0 / 3.0)) ** (vcycle_ms / ms_step)),
            },
            "roofline": {
                "bound": "hbm", "kernel": "fac_kernel (persistent AlgFAC, a3-a10)", "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": model_bytes, "stream_bytes_per_launch": stream_bytes,
                "stream_gbs": stream_bytes / (fac_avg_ms * 1e-3) / 1e9, "launch_ms": fac_avg_ms,
                # the matrix entries themselves at this build's widths (8-byte value + 2- or 4-byte column), no padding, no headers
                "useful_bytes": useful_bytes, "useful_gbs": useful_bytes / (fac_avg_ms * 1e-3) / 1e9,
                "traffic": traffic,
                # DRAM bytes of the committed ncu capture of THIS kernel source / the launch time measured now / peak
                "frac_dram": (traffic / (fac_avg_ms * 1e-3) / 1e9 / peak) if traffic else None,
                "frac_stream": stream_bytes / (fac_avg_ms * 1e-3) / 1e9 / peak,
                "kernel_source_hash": kernel_source_hash(),
            },
        }
        if os.environ.get("AMGDD_FAC_PROFILE", "0") == "1":
            # debugging aid (never a timed run): SM cycles of every step of the AlgFAC program, thread 0 of every CTA, over the cycles
            # of the per-launch timing loop above; shares by step kind and by level
            ops = fac_ops
            tot = float(sum(o[2] + o[3] for o in ops)) or 1.0
            by_kind, by_level = {}, {}
            for kind, lvl, cyc, bar, ring, opw in ops:
                by_kind[kind] = by_kind.get(kind, 0.0) + (cyc + bar) / tot
                by_level[str(lvl)] = by_level.get(str(lvl), 0.0) + (cyc + bar) / tot
            line["fac_step_profile"] = {
                "cycles_per_subdomain_and_cycle": tot / (args.steps * p.num_subdomains), "share_by_kind": by_kind, "share_by_level": by_level,
                "steps": [{"kind": k, "level": l, "cycles": c / (args.steps * p.num_subdomains), "barrier": bw / (args.steps * p.num_subdomains),
                           "ring_wait": rw / (args.steps * p.num_subdomains), "operand_wait": ow / (args.steps * p.num_subdomains)}
                          for k, l, c, bw, rw, ow in ops]}
        if not args.no_cpu_baseline or not args.no_per_config:
            m.amgdd_destroy(h)
            del b, x
            torch.cuda.empty_cache()
        if not args.no_per_config and not distributed and args.config == 4 and args.scale is None and args.eta is None and not args.smoother:
            # the other BASELINE.json configs, a few seconds each (config 3 needs 112 GB and a long setup: --all-configs)
            line["per_config"] = {}
            for cfg, eta in [(1, None), (2, None), (5, None)] + ([(3, 1)] if args.all_configs else []):
                name, rec = measure_config(m, torch, cfg, max(args.steps, 10), args.warmup, eta)
                line["per_config"][name] = rec
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_time_per_cycle(p, args.cpu_sample or default_cpu_sample(p), 3, 1, args.smoother)
        print(json.dumps(line))
    if distributed:
        dist.barrier()
        dist.destroy_process_group()


def run_sharded(args, p, rank, world, local_rank, m, torch, dist):
    """--shard: the subdomains are split over the ranks (contiguous blocks); one step = one AMG-DD cycle of the whole problem
    with the staged exchange of include/amgdd.h ("sharding over ranks") over torch.distributed.  Strong scaling: the total
    work is fixed.  Built and tested with virtual ranks on one GPU (tests/test_gpu_sharded.py); never timed on several GPUs."""
    from paper_1906_10575_b200.sharded import DistComm, allgather_cycle, setup_exchange, sharded_cycle
    if not dist.is_initialized():
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    t0 = time.time()
    h = m.amgdd_setup_shard(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.num_ghost, p.max_levels, p.theta,
                            p.coarse_max, rank=rank, nranks=world)
    comm = DistComm()
    setup_exchange({rank: h}, comm)
    setup_s = time.time() - t0
    stream = torch.cuda.current_stream()
    m.amgdd_set_stream(h, stream)
    b = {rank: torch.from_numpy(p.b).cuda()}
    x = {rank: torch.zeros(p.n, dtype=torch.float64, device="cuda")}
    nfac, nu = p.num_fac_cycles, p.relax_sweeps
    cycle = (lambda want=False: sharded_cycle({rank: h}, b, x, comm, nfac, nu, want_norm=want)) if args.shard == "alg5" else \
            (lambda want=False: allgather_cycle({rank: h}, b, x, comm, nfac, nu)[rank])
    nlev = m.amgdd_num_levels(h)
    norms = [cycle(True) for _ in range(p.num_cycles)]
    for _ in range(args.warmup):
        cycle()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier(); torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(args.steps):
        cycle()
    e1.record(stream)
    dist.barrier(); torch.cuda.synchronize()
    ms = torch.tensor([e0.elapsed_time(e1) / args.steps], dtype=torch.float64, device="cuda")
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": float(ms.item()), "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": float(ms.item()), "higher_is_better": False, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": workload_name(p, args), "subdomains": p.num_subdomains, "multi_gpu": f"sharded over {world} ranks, exchange {args.shard}",
                       "setup_seconds": setup_s, "note": "NEXT 4; unmeasured on multi-GPU hardware before this run"},
            "residual_norms_at_cycle_start": norms,
            # per cycle: r_l on the owned rows of L + 1 levels (+ the sum of squares), a gather and a scatter per stage, AlgFAC
            "gpu_launches": int(((nlev + 1) + 2 * (2 * nlev) + 1) * args.steps)}))
    dist.barrier()
    dist.destroy_process_group()


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference" and rank != 0:
        return
    import workloads as wl
    p = wl.make_config(args.config, args.scale, eta=args.eta)
    if args.impl == "reference":
        run_reference(args, p, rank, world)
    else:
        run_b200(args, p, rank, world, local_rank)


if __name__ == "__main__":
    main()
