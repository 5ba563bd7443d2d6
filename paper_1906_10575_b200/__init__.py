"""paper_1906_10575_b200 -- B200-native AMG-DD local-solve hot path (arXiv 1906.10575).

Thin Python binding of the C ABI in include/amgdd.h (same names, argument marshalling only).
Every step of the path runs in the hand-written CUDA kernels of libamgdd.so; PyTorch supplies
device memory and streams.  There is no CPU fallback: if libamgdd.so cannot be loaded the import
fails, and without a CUDA device amgdd_setup returns AMGDD_ERR_CUDA.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

_vp, _i32, _i64, _f64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double

EXPORTS = [
    "amgdd_setup", "amgdd_solve", "amgdd_solve_host", "amgdd_vcycle", "amgdd_residual_norm", "amgdd_residual_norm_static", "amgdd_set_smoother", "amgdd_set_stream", "amgdd_destroy",
    "amgdd_strerror", "amgdd_last_error_detail", "amgdd_num_levels", "amgdd_level_size", "amgdd_get_cf",
    "amgdd_get_level_matrix", "amgdd_composite_size", "amgdd_get_composite", "amgdd_get_stats",
    "amgdd_last_solve_profile", "amgdd_pack_stream", "amgdd_debug_fac_cycles", "amgdd_debug_fac_op_cycles",
    "amgdd_debug_read_block",
    "amgdd_setup_shard", "amgdd_shard_plan_create", "amgdd_shard_plan_destroy", "amgdd_get_shard_plan", "amgdd_shard_plan_info",
    "amgdd_shard_plan_level", "amgdd_shard_plan_owner_rank", "amgdd_shard_plan_list", "amgdd_shard_plan_stage_vector",
    "amgdd_shard_plan_recv_filter", "amgdd_shard_plan_apply_drop", "amgdd_shard_commit", "amgdd_shard_stage_counts",
    "amgdd_shard_stage_pack", "amgdd_shard_stage_unpack", "amgdd_shard_local_solve", "amgdd_shard_sqnorm",
    "amgdd_shard_owned_count", "amgdd_shard_pack_owned", "amgdd_shard_unpack_owned",
]


class AmgddStats(ctypes.Structure):
    _fields_ = [
        ("num_levels", _i32), ("num_subdomains", _i32), ("n_fine", _i64), ("nnz_hierarchy", _i64),
        ("nnz_composite_real", _i64), ("overhead", _f64), ("operator_complexity", _f64), ("sum_real", _i64),
        ("sum_ghost", _i64), ("dropped_interp_entries", _i64), ("device_bytes", _i64),
        ("shared_level_instances", _i64), ("model_bytes_fac_iter", _f64 * 2), ("stream_bytes_fac_iter", _f64 * 2),
        ("model_bytes_global", _f64), ("setup_seconds_hierarchy", _f64), ("setup_seconds_composite", _f64),
        ("block_bytes", _i32), ("num_ways", _i32), ("window", _i32), ("ring_stages", _i32), ("x_cap", _i32), ("fac_grid", _i32), ("fac_block", _i32),
        ("fac_smem_bytes", _i32), ("max_n_bar", _i64),
        ("assembled_on_device", _i32), ("index_sets_on_device", _i32), ("setup_seconds_index_sets", _f64),
        ("setup_seconds_assembly", _f64), ("setup_seconds_upload", _f64),
        ("useful_bytes_fac_iter", _f64 * 2),
    ]


class AmgddError(RuntimeError):
    def __init__(self, code, what, detail):
        super().__init__(f"{what} (status {code}): {detail}")
        self.code = code


def _load():
    lib_path = _build.LIB
    if _build.needs_build():
        # (re)building is not a fallback: it produces the same CUDA library or raises
        _build.build()
    L = ctypes.CDLL(lib_path)
    L.amgdd_setup.argtypes = [_i64, _vp, _vp, _vp, _i32, _vp, _i32, _i32, _i32, _f64, _i32, ctypes.POINTER(_vp)]
    L.amgdd_solve.argtypes = [_vp, _vp, _vp, _i32, _i32, _i32, _vp]
    L.amgdd_solve_host.argtypes = [_vp, _vp, _vp, _i32, _i32, _i32, _vp]
    L.amgdd_residual_norm.argtypes = [_vp, _vp, _vp, _vp]
    L.amgdd_residual_norm_static.argtypes = [_i64, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
    L.amgdd_vcycle.argtypes = [_vp, _vp, _vp, _i32, _i32, _i32, _vp]
    L.amgdd_set_stream.argtypes = [_vp, _vp]
    L.amgdd_set_smoother.argtypes = [_vp, _i32]
    L.amgdd_destroy.argtypes = [_vp]
    L.amgdd_strerror.restype = ctypes.c_char_p
    L.amgdd_strerror.argtypes = [ctypes.c_int]
    L.amgdd_last_error_detail.restype = ctypes.c_char_p
    L.amgdd_num_levels.argtypes = [_vp, _vp]
    L.amgdd_level_size.argtypes = [_vp, _i32, _vp, _vp, _vp]
    L.amgdd_get_cf.argtypes = [_vp, _i32, _vp]
    L.amgdd_get_level_matrix.argtypes = [_vp, _i32, _i32, _vp, _vp, _vp]
    L.amgdd_composite_size.argtypes = [_vp, _i32, _i32, _vp, _vp]
    L.amgdd_get_composite.argtypes = [_vp, _i32, _i32, _vp, _vp]
    L.amgdd_get_stats.argtypes = [_vp, ctypes.POINTER(AmgddStats)]
    L.amgdd_last_solve_profile.argtypes = [_vp, _vp, _vp]
    L.amgdd_debug_fac_cycles.argtypes = [_vp, _vp, _i32]
    L.amgdd_debug_fac_op_cycles.argtypes = [_vp, _vp, _i32, _vp]
    L.amgdd_debug_read_block.argtypes = [_vp, _i32, _i32, _i32, _vp, _i64, _vp]
    L.amgdd_pack_stream.argtypes = [_i32, _i32, _vp, _vp, _vp, _vp, _i32, _i32, _vp, _i64, _vp, _vp]
    L.amgdd_setup_shard.argtypes = [_i64, _vp, _vp, _vp, _i32, _vp, _i32, _i32, _i32, _f64, _i32, _i32, _i32, ctypes.POINTER(_vp)]
    L.amgdd_shard_plan_create.argtypes = [_i64, _vp, _vp, _vp, _i32, _vp, _i32, _i32, _f64, _i32, _i32, _i32, ctypes.POINTER(_vp)]
    L.amgdd_shard_plan_destroy.argtypes = [_vp]
    L.amgdd_get_shard_plan.argtypes = [_vp, ctypes.POINTER(_vp)]
    L.amgdd_shard_plan_info.argtypes = [_vp, _vp]
    L.amgdd_shard_plan_level.argtypes = [_vp, _i32, _vp, _vp, _vp]
    L.amgdd_shard_plan_owner_rank.argtypes = [_vp, _i32, _vp]
    L.amgdd_shard_plan_list.argtypes = [_vp, _i32, _i32, _i32, _vp, _vp]
    L.amgdd_shard_plan_stage_vector.argtypes = [_vp, _i32, _vp]
    L.amgdd_shard_plan_recv_filter.argtypes = [_vp, _i32, _i32, _vp, _i64, _vp, _vp]
    L.amgdd_shard_plan_apply_drop.argtypes = [_vp, _i32, _i32, _vp, _i64]
    L.amgdd_shard_commit.argtypes = [_vp]
    L.amgdd_shard_stage_counts.argtypes = [_vp, _i32, _vp, _vp]
    L.amgdd_shard_stage_pack.argtypes = [_vp, _i32, _vp, _vp, _vp]
    L.amgdd_shard_stage_unpack.argtypes = [_vp, _i32, _vp, _vp]
    L.amgdd_shard_local_solve.argtypes = [_vp, _vp, _i32, _i32]
    L.amgdd_shard_sqnorm.argtypes = [_vp, _vp]
    L.amgdd_shard_owned_count.argtypes = [_vp, _i32, _vp]
    L.amgdd_shard_pack_owned.argtypes = [_vp, _vp, _vp]
    L.amgdd_shard_unpack_owned.argtypes = [_vp, _i32, _vp, _vp]
    return L


lib = _load()


def _check(rc):
    if rc != 0:
        raise AmgddError(rc, lib.amgdd_strerror(rc).decode(), lib.amgdd_last_error_detail().decode())


def amgdd_strerror(code: int) -> str:
    return lib.amgdd_strerror(code).decode()


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


class Handle:
    """Owner of an amgdd_handle_t."""

    def __init__(self, ptr):
        self._h = ptr

    def __del__(self):
        self.destroy()

    def destroy(self):
        if getattr(self, "_h", None) and lib is not None:       # lib is None during interpreter shutdown
            lib.amgdd_destroy(self._h)
        self._h = None


def amgdd_setup(n, rowptr, colind, vals, num_subdomains, owner, eta, num_ghost=1, max_levels=25, theta=0.25,
                coarse_max=64) -> Handle:
    """amgdd_setup of include/amgdd.h; numpy (host) arrays in, Handle out."""
    rowptr = None if rowptr is None else _np(rowptr, np.int64)
    colind = None if colind is None else _np(colind, np.int32)
    vals = None if vals is None else _np(vals, np.float64)
    owner = None if owner is None else _np(owner, np.int32)
    ptr = lambda a: None if a is None else a.ctypes.data
    out = _vp()
    _check(lib.amgdd_setup(n, ptr(rowptr), ptr(colind), ptr(vals), num_subdomains, ptr(owner), eta, num_ghost,
                           max_levels, theta, coarse_max, ctypes.byref(out)))
    return Handle(out.value)


def _dev_ptr(t, n):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() >= n):
        raise TypeError("expected a contiguous float64 CUDA tensor of length >= n")
    return t.data_ptr()


SMOOTHER_L1_JACOBI, SMOOTHER_CF_L1_JACOBI = 0, 1


def amgdd_set_smoother(h: Handle, kind: int):
    """amgdd_set_smoother: 0 l1-Jacobi (default), 1 CF l1-Jacobi."""
    _check(lib.amgdd_set_smoother(h._h, int(kind)))


def amgdd_set_stream(h: Handle, stream=None):
    """Use a torch.cuda.Stream (default: torch's current stream)."""
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    _check(lib.amgdd_set_stream(h._h, s.cuda_stream))
    h._stream = int(s.cuda_stream)                   # remembered for the stream check of sharded.py (0 / absent: legacy default stream)


def amgdd_solve(h: Handle, b, x, num_cycles, num_fac_cycles=2, relax_sweeps=1, want_norms=True):
    """amgdd_solve: b, x float64 CUDA tensors (x in/out).  Returns resnorm[0..num_cycles] or None."""
    n = amgdd_level_size(h, 0)[0]
    res = np.empty(num_cycles + 1, dtype=np.float64) if want_norms else None
    _check(lib.amgdd_solve(h._h, _dev_ptr(b, n), _dev_ptr(x, n), num_cycles, num_fac_cycles, relax_sweeps,
                           res.ctypes.data if want_norms else None))
    return res


def amgdd_solve_host(h: Handle, b_host, x_host, num_cycles, num_fac_cycles=2, relax_sweeps=1):
    """amgdd_solve_host: numpy (or pinned torch CPU) float64 arrays, x_host updated in place."""
    def ptr(a):
        if isinstance(a, np.ndarray):
            assert a.dtype == np.float64 and a.flags.c_contiguous
            return a.ctypes.data
        return a.data_ptr()
    res = np.empty(num_cycles + 1, dtype=np.float64)
    _check(lib.amgdd_solve_host(h._h, ptr(b_host), ptr(x_host), num_cycles, num_fac_cycles, relax_sweeps, res.ctypes.data))
    return res


def amgdd_vcycle(h: Handle, b, x, num_cycles, nu1=1, nu2=1, want_norms=True):
    """amgdd_vcycle: AMG V(nu1,nu2)-cycles (Alg. 1) on the handle's hierarchy; b, x float64 CUDA tensors."""
    n = amgdd_level_size(h, 0)[0]
    res = np.empty(num_cycles + 1, dtype=np.float64) if want_norms else None
    _check(lib.amgdd_vcycle(h._h, _dev_ptr(b, n), _dev_ptr(x, n), num_cycles, nu1, nu2, res.ctypes.data if want_norms else None))
    return res


def amgdd_residual_norm(h: Handle, b, x) -> float:
    n = amgdd_level_size(h, 0)[0]
    out = _f64()
    _check(lib.amgdd_residual_norm(h._h, _dev_ptr(b, n), _dev_ptr(x, n), ctypes.byref(out)))
    return out.value


STATIC_MAX_ROWS = 16777216


def amgdd_residual_norm_static(n, rowptr, colind, vals, b, x, out_norm, r=None, stream=None):
    """amgdd_residual_norm_static: || b - A x ||_2 without any device allocation, for callers that cannot
    allocate where they need the norm (all device memory already in a pool, no handle, no room for the
    synchronisation of cudaFree).  Everything is a CUDA tensor on the current device that the CALLER made:
    rowptr int64 [n+1], colind int32, vals / b / x float64, out_norm float64 [1] (written asynchronously on
    `stream`, default torch's current stream: synchronise before reading it), r float64 [n] or None.  At most
    STATIC_MAX_ROWS rows (the scratch is a fixed 512 KiB device array inside the library); concurrent calls on
    one device race on that array.  The first call on a device should be made before any stream capture."""
    import torch

    def ptr(t, dt, count, name):
        if t is None:
            return None
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() >= count):
            raise TypeError(f"{name}: expected a contiguous {dt} CUDA tensor with at least {count} entries")
        return t.data_ptr()
    n = int(n)
    big = n > STATIC_MAX_ROWS or n <= 0          # the library reports these; do not touch the tensors' sizes first
    nnz = 0 if big else int(colind.numel())
    s = stream if stream is not None else torch.cuda.current_stream()
    _check(lib.amgdd_residual_norm_static(
        n, ptr(rowptr, torch.int64, 0 if big else n + 1, "rowptr"), ptr(colind, torch.int32, nnz, "colind"),
        ptr(vals, torch.float64, nnz, "vals"), ptr(b, torch.float64, 0 if big else n, "b"),
        ptr(x, torch.float64, 0 if big else n, "x"), ptr(r, torch.float64, 0 if big else n, "r"),
        ptr(out_norm, torch.float64, 1, "out_norm"), s.cuda_stream))


def amgdd_destroy(h: Handle):
    h.destroy()


def amgdd_num_levels(h: Handle) -> int:
    out = _i32()
    _check(lib.amgdd_num_levels(h._h, ctypes.byref(out)))
    return out.value


def amgdd_level_size(h: Handle, l: int):
    n, a, p = _i64(), _i64(), _i64()
    _check(lib.amgdd_level_size(h._h, l, ctypes.byref(n), ctypes.byref(a), ctypes.byref(p)))
    return n.value, a.value, p.value


def amgdd_get_cf(h: Handle, l: int) -> np.ndarray:
    out = np.empty(amgdd_level_size(h, l)[0], dtype=np.int8)
    _check(lib.amgdd_get_cf(h._h, l, out.ctypes.data))
    return out


def amgdd_get_level_matrix(h: Handle, l: int, which: int):
    n, nnzA, nnzP = amgdd_level_size(h, l)
    nnz = nnzA if which == 0 else nnzP
    rp, ci, v = np.empty(n + 1, np.int64), np.empty(nnz, np.int32), np.empty(nnz, np.float64)
    _check(lib.amgdd_get_level_matrix(h._h, l, which, rp.ctypes.data, ci.ctypes.data, v.ctypes.data))
    return rp, ci, v


def amgdd_composite_size(h: Handle, p: int, l: int):
    nr, ng = _i64(), _i64()
    _check(lib.amgdd_composite_size(h._h, p, l, ctypes.byref(nr), ctypes.byref(ng)))
    return nr.value, ng.value


def amgdd_get_composite(h: Handle, p: int, l: int):
    nr, ng = amgdd_composite_size(h, p, l)
    real, ghost = np.empty(nr, np.int32), np.empty(ng, np.int32)
    _check(lib.amgdd_get_composite(h._h, p, l, real.ctypes.data, ghost.ctypes.data))
    return real, ghost


def amgdd_get_stats(h: Handle) -> dict:
    s = AmgddStats()
    _check(lib.amgdd_get_stats(h._h, ctypes.byref(s)))
    d = {}
    for name, _ in AmgddStats._fields_:
        v = getattr(s, name)
        d[name] = list(v) if hasattr(v, "__len__") else v
    return d


NUM_WAYS = 16
GROUP_BYTES_NARROW, GROUP_BYTES_WIDE, HEADER_BYTES_NARROW, HEADER_BYTES_WIDE = 1280, 1536, 128, 256
WAY_DTYPE = np.dtype([("grp_off128", np.uint32), ("hdr_off128", np.uint32), ("ngroups", np.uint32), ("ngroups_real", np.uint32),
                      ("nslices", np.uint32), ("nslices_real", np.uint32), ("reserved", np.uint32, (2,))])


def amgdd_pack_stream(rowptr, colind, vals, wide=False, n_real=None, window=256, row_flags=None):
    """amgdd_pack_stream: CSR (host) -> (bytes of the packed SELL-32 group streams as a uint8 array, the
    NUM_WAYS way descriptors as a structured array)."""
    rowptr = _np(rowptr, np.int32)
    colind = _np(colind, np.int32)
    vals = _np(vals, np.float64)
    row_flags = None if row_flags is None else _np(row_flags, np.uint8)
    nrows = len(rowptr) - 1
    n_real = nrows if n_real is None else n_real
    nbytes = _i64()
    ways = np.zeros(NUM_WAYS, dtype=WAY_DTYPE)
    args = (nrows, n_real, rowptr.ctypes.data, colind.ctypes.data, vals.ctypes.data,
            None if row_flags is None else row_flags.ctypes.data, int(wide), window)
    _check(lib.amgdd_pack_stream(*args, None, 0, ctypes.byref(nbytes), ways.ctypes.data))
    out = np.zeros(max(nbytes.value, 1), dtype=np.uint8)
    _check(lib.amgdd_pack_stream(*args, out.ctypes.data, nbytes.value, ctypes.byref(nbytes), ways.ctypes.data))
    return out[:nbytes.value], ways


FAC_CYCLE_NAMES = ["sync", "fetch_subdomain", "pre_actions", "matvec_startup", "total", "gather_a3", "first0", "op_relax", "op_At",
                   "op_restrict", "op_recalc", "op_interp", "coarse", "update_a10", "wait_slice_operands", "wait_ring_block"]


def amgdd_debug_fac_cycles(h: Handle, reset=True) -> dict:
    """Per-phase SM cycles of the AlgFAC kernel summed over its CTAs (needs AMGDD_FAC_PROFILE=1 at setup)."""
    out = (ctypes.c_int64 * 16)()
    _check(lib.amgdd_debug_fac_cycles(h._h, out, int(reset)))
    return dict(zip(FAC_CYCLE_NAMES, [int(v) for v in out]))


OP_KIND_NAMES = ["begin", "first0", "relax", "At", "restrict", "recalc", "interp", "coarse", "end"]


def amgdd_debug_fac_op_cycles(h: Handle, n=256):
    """Per-step SM cycles of the AlgFAC program (needs AMGDD_FAC_PROFILE=1 at setup): list of
    (kind name, level, step cycles, barrier-wait cycles, ring-wait cycles, slice-operand-wait cycles)."""
    out = np.zeros(4 * n, dtype=np.int64)
    kl = np.full(n, -1, dtype=np.int32)
    _check(lib.amgdd_debug_fac_op_cycles(h._h, out.ctypes.data, n, kl.ctypes.data))
    return [(OP_KIND_NAMES[k // 256], int(k % 256), int(out[j]), int(out[n + j]), int(out[2 * n + j]), int(out[3 * n + j]))
            for j, k in enumerate(kl) if k >= 0]


BLOCK_ARRAYS = {"gid": 0, "dinv": 1, "A": 2, "P": 3, "R": 4, "owned": 5}


def amgdd_debug_read_block(h: Handle, p: int, level: int, which: str) -> np.ndarray:
    """One array of a private (subdomain, level) block as the device holds it (bytes; empty for a shared level)."""
    nbytes = _i64(0)
    w = BLOCK_ARRAYS[which]
    _check(lib.amgdd_debug_read_block(h._h, p, level, w, None, 0, ctypes.byref(nbytes)))
    out = np.zeros(nbytes.value, dtype=np.uint8)
    if nbytes.value:
        _check(lib.amgdd_debug_read_block(h._h, p, level, w, out.ctypes.data, nbytes.value, ctypes.byref(nbytes)))
    return out


def amgdd_last_solve_profile(h: Handle):
    ms = (ctypes.c_double * 4)()
    ln = (ctypes.c_int64 * 3)()
    _check(lib.amgdd_last_solve_profile(h._h, ms, ln))
    return {"ms_residual": ms[0], "ms_restrict": ms[1], "ms_fac": ms[2], "ms_total": ms[3],
            "launches": [int(ln[0]), int(ln[1]), int(ln[2])]}


# ---- sharding over ranks (include/amgdd.h, "sharding over ranks"; the exchange driver is in sharded.py) ----
class ShardPlan:
    """An amgdd_shard_plan_t: owned (amgdd_shard_plan_create, host only) or borrowed from a Handle."""

    def __init__(self, ptr, owned, keep=None):
        self._p, self._owned, self._keep = ptr, owned, keep

    def __del__(self):
        if getattr(self, "_p", None) and self._owned and lib is not None:
            lib.amgdd_shard_plan_destroy(self._p)
        self._p = None


def amgdd_setup_shard(n, rowptr, colind, vals, num_subdomains, owner, eta, num_ghost=1, max_levels=25, theta=0.25,
                      coarse_max=64, rank=0, nranks=1) -> Handle:
    rowptr, colind, vals, owner = _np(rowptr, np.int64), _np(colind, np.int32), _np(vals, np.float64), _np(owner, np.int32)
    out = _vp()
    _check(lib.amgdd_setup_shard(n, rowptr.ctypes.data, colind.ctypes.data, vals.ctypes.data, num_subdomains, owner.ctypes.data,
                                 eta, num_ghost, max_levels, theta, coarse_max, rank, nranks, ctypes.byref(out)))
    return Handle(out.value)


def amgdd_shard_plan_create(n, rowptr, colind, vals, num_subdomains, owner, eta, max_levels=25, theta=0.25, coarse_max=64,
                            rank=0, nranks=1) -> ShardPlan:
    rowptr, colind, vals, owner = _np(rowptr, np.int64), _np(colind, np.int32), _np(vals, np.float64), _np(owner, np.int32)
    out = _vp()
    _check(lib.amgdd_shard_plan_create(n, rowptr.ctypes.data, colind.ctypes.data, vals.ctypes.data, num_subdomains,
                                       owner.ctypes.data, eta, max_levels, theta, coarse_max, rank, nranks, ctypes.byref(out)))
    return ShardPlan(out.value, True)


def amgdd_get_shard_plan(h: Handle) -> ShardPlan:
    out = _vp()
    _check(lib.amgdd_get_shard_plan(h._h, ctypes.byref(out)))
    return ShardPlan(out.value, False, keep=h)


def amgdd_shard_plan_info(p: ShardPlan) -> dict:
    a = np.zeros(6, dtype=np.int32)
    _check(lib.amgdd_shard_plan_info(p._p, a.ctypes.data))
    return dict(zip(["rank", "nranks", "num_levels", "num_stages", "sub_lo", "sub_hi"], [int(v) for v in a]))


def amgdd_shard_plan_level(p: ShardPlan, l: int):
    n, off, no = _i64(), _i64(), _i64()
    _check(lib.amgdd_shard_plan_level(p._p, l, ctypes.byref(n), ctypes.byref(off), ctypes.byref(no)))
    return n.value, off.value, no.value


def amgdd_shard_plan_owner_rank(p: ShardPlan, l: int) -> np.ndarray:
    out = np.empty(amgdd_shard_plan_level(p, l)[0], dtype=np.int32)
    _check(lib.amgdd_shard_plan_owner_rank(p._p, l, out.ctypes.data))
    return out


def amgdd_shard_plan_list(p: ShardPlan, which: int, stage: int, peer: int) -> np.ndarray:
    cnt = _i64()
    _check(lib.amgdd_shard_plan_list(p._p, which, stage, peer, None, ctypes.byref(cnt)))
    out = np.empty(cnt.value, dtype=np.int64)
    if cnt.value:
        _check(lib.amgdd_shard_plan_list(p._p, which, stage, peer, out.ctypes.data, ctypes.byref(cnt)))
    return out


def amgdd_shard_plan_stage_vector(p: ShardPlan, stage: int) -> int:
    v = _i32()
    _check(lib.amgdd_shard_plan_stage_vector(p._p, stage, ctypes.byref(v)))
    return v.value


def amgdd_shard_plan_recv_filter(p: ShardPlan, stage: int, src: int, announced) -> np.ndarray:
    announced = _np(announced, np.int64)
    red = np.empty(max(1, len(announced)), dtype=np.int64)
    nred = _i64()
    _check(lib.amgdd_shard_plan_recv_filter(p._p, stage, src, announced.ctypes.data if len(announced) else None, len(announced),
                                            red.ctypes.data, ctypes.byref(nred)))
    return red[:nred.value].copy()


def amgdd_shard_plan_apply_drop(p: ShardPlan, stage: int, dest: int, redundant):
    redundant = _np(redundant, np.int64)
    _check(lib.amgdd_shard_plan_apply_drop(p._p, stage, dest, redundant.ctypes.data if len(redundant) else None, len(redundant)))


def amgdd_shard_commit(h: Handle):
    _check(lib.amgdd_shard_commit(h._h))


def amgdd_shard_stage_counts(h: Handle, stage: int, nranks: int):
    s, r = np.zeros(nranks, dtype=np.int64), np.zeros(nranks, dtype=np.int64)
    _check(lib.amgdd_shard_stage_counts(h._h, stage, s.ctypes.data, r.ctypes.data))
    return s, r


def amgdd_shard_stage_pack(h: Handle, stage: int, b, x, sendbuf):
    n = amgdd_level_size(h, 0)[0]
    _check(lib.amgdd_shard_stage_pack(h._h, stage, _dev_ptr(b, n), _dev_ptr(x, n), sendbuf.data_ptr() if sendbuf is not None and sendbuf.numel() else None))


def amgdd_shard_stage_unpack(h: Handle, stage: int, x, recvbuf):
    n = amgdd_level_size(h, 0)[0]
    _check(lib.amgdd_shard_stage_unpack(h._h, stage, _dev_ptr(x, n), recvbuf.data_ptr() if recvbuf is not None and recvbuf.numel() else None))


def amgdd_shard_local_solve(h: Handle, x, num_fac_cycles=2, relax_sweeps=1):
    n = amgdd_level_size(h, 0)[0]
    _check(lib.amgdd_shard_local_solve(h._h, _dev_ptr(x, n), num_fac_cycles, relax_sweeps))


def amgdd_shard_sqnorm(h: Handle) -> float:
    out = _f64()
    _check(lib.amgdd_shard_sqnorm(h._h, ctypes.byref(out)))
    return out.value


def amgdd_shard_owned_count(h: Handle, rank: int) -> int:
    out = _i64()
    _check(lib.amgdd_shard_owned_count(h._h, rank, ctypes.byref(out)))
    return out.value


def amgdd_shard_pack_owned(h: Handle, x, buf):
    n = amgdd_level_size(h, 0)[0]
    _check(lib.amgdd_shard_pack_owned(h._h, _dev_ptr(x, n), buf.data_ptr()))


def amgdd_shard_unpack_owned(h: Handle, src_rank: int, buf, x):
    n = amgdd_level_size(h, 0)[0]
    _check(lib.amgdd_shard_unpack_owned(h._h, src_rank, buf.data_ptr(), _dev_ptr(x, n)))


def amgdd_shard_plan_destroy(p: ShardPlan):
    """Frees a plan made by amgdd_shard_plan_create (borrowed plans are left alone)."""
    if p._p and p._owned:
        lib.amgdd_shard_plan_destroy(p._p)
    p._p = None
