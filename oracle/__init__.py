"""ctypes binding of the CPU oracle (oracle/amgdd_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg.  The product package never imports this module.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "amgdd_oracle.cpp")
_SO = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _SO])
    return _SO


_lib = None
_vp, _i32, _i64, _f64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double


def _load():
    global _lib
    if _lib is not None:
        return _lib
    L = ctypes.CDLL(build())
    L.orc_create.restype = _vp
    L.orc_create.argtypes = [_i64, _vp, _vp, _vp, _f64, _i32, _i32, _vp]
    L.orc_destroy.argtypes = [_vp]
    L.orc_set_smoother.argtypes = [_vp, _i32]
    L.orc_num_levels.argtypes = [_vp]
    L.orc_level_size.argtypes = [_vp, _i32, _vp, _vp, _vp]
    L.orc_get_cf.argtypes = [_vp, _i32, _vp]
    L.orc_get_matrix.argtypes = [_vp, _i32, _i32, _vp, _vp, _vp]
    L.orc_get_dinv.argtypes = [_vp, _i32, _vp]
    L.orc_set_level_values.argtypes = [_vp, _i32, _vp]
    L.orc_set_partition.argtypes = [_vp, _i32, _vp, _i32, _i32]
    L.orc_composite_size.argtypes = [_vp, _i32, _i32, _vp, _vp]
    L.orc_get_composite.argtypes = [_vp, _i32, _i32, _vp, _vp]
    L.orc_cycle.argtypes = [_vp, _vp, _vp, _i32, _i32, _vp, _i32, _i32]
    L.orc_residual_norm.restype = _f64
    L.orc_residual_norm.argtypes = [_vp, _vp, _vp]
    L.orc_solve.argtypes = [_vp, _vp, _vp, _i32, _i32, _i32, _vp, _i32]
    L.orc_fac_local.argtypes = [_vp, _i32, _vp, _i32, _i32, _vp]
    L.orc_relax.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp, _i32]
    L.orc_vcycle.argtypes = [_vp, _vp, _vp, _i32, _i32]
    L.orc_coarse_solve.argtypes = [_vp, _vp]
    L.orc_counters.argtypes = [_vp, _vp]
    L.orc_dropped.restype = _i64
    L.orc_dropped.argtypes = [_vp]
    L.orc_overhead.restype = _f64
    L.orc_overhead.argtypes = [_vp, _i32]
    L.orc_max_threads.restype = _i32
    _lib = L
    return L


def _p(a):
    return a.ctypes.data if a is not None else None


class Oracle:
    """AMG hierarchy (S1-S5, S8) + composite grids (S6, S7) + AMG-DD cycles (Alg. 2 / Alg. 4)."""

    def __init__(self, n, rowptr, colind, vals, theta, max_levels=25, coarse_max=64):
        L = _load()
        rowptr = np.ascontiguousarray(rowptr, dtype=np.int64)
        colind = np.ascontiguousarray(colind, dtype=np.int32)
        vals = np.ascontiguousarray(vals, dtype=np.float64)
        err = ctypes.c_int(0)
        self._h = L.orc_create(n, _p(rowptr), _p(colind), _p(vals), theta, max_levels, coarse_max, ctypes.byref(err))
        if not self._h:
            raise RuntimeError(f"oracle setup failed with code {err.value}")
        self.n = n
        self.num_levels = L.orc_num_levels(self._h)
        self.num_subdomains = 0

    def __del__(self):
        if getattr(self, "_h", None):
            _load().orc_destroy(self._h)
            self._h = None

    def set_smoother(self, kind):
        """0: l1-Jacobi (BASELINE), 1: CF l1-Jacobi: C- then F-points before, F- then C-points after the coarse correction."""
        _load().orc_set_smoother(self._h, int(kind))

    # ---- hierarchy introspection ----
    def level_size(self, l):
        n, a, p = _i64(), _i64(), _i64()
        _load().orc_level_size(self._h, l, ctypes.byref(n), ctypes.byref(a), ctypes.byref(p))
        return n.value, a.value, p.value

    def cf(self, l):
        n, _, _ = self.level_size(l)
        out = np.empty(n, dtype=np.int8)
        _load().orc_get_cf(self._h, l, _p(out))
        return out

    def matrix(self, l, which):
        """which = 'A' or 'P' -> (rowptr, colind, vals)."""
        n, nnzA, nnzP = self.level_size(l)
        nnz = nnzA if which == "A" else nnzP
        rp = np.empty(n + 1, dtype=np.int64)
        ci = np.empty(nnz, dtype=np.int32)
        v = np.empty(nnz, dtype=np.float64)
        _load().orc_get_matrix(self._h, l, 0 if which == "A" else 1, _p(rp), _p(ci), _p(v))
        return rp, ci, v

    def scipy_matrix(self, l, which):
        import scipy.sparse as sp
        rp, ci, v = self.matrix(l, which)
        n = self.level_size(l)[0]
        m = n if which == "A" else self.level_size(l + 1)[0]
        return sp.csr_matrix((v, ci, rp), shape=(n, m))

    def dinv(self, l):
        out = np.empty(self.level_size(l)[0], dtype=np.float64)
        _load().orc_get_dinv(self._h, l, _p(out))
        return out

    def set_level_values(self, l, vals):
        """Test support (no arithmetic of the method): overwrite the values of A_l, l >= 1, on its stored pattern; the l1
        diagonal and, on the coarsest level, the LU are refreshed."""
        vals = np.ascontiguousarray(vals, dtype=np.float64)
        assert vals.shape == (self.level_size(l)[1],)
        rc = _load().orc_set_level_values(self._h, l, _p(vals))
        if rc != 0:
            raise RuntimeError(f"orc_set_level_values failed with {rc}")

    # ---- decomposition ----
    def set_partition(self, num_subdomains, owner, eta, num_ghost=1):
        owner = np.ascontiguousarray(owner, dtype=np.int32)
        rc = _load().orc_set_partition(self._h, num_subdomains, _p(owner), eta, num_ghost)
        if rc != 0:
            raise RuntimeError(f"oracle set_partition failed with code {rc}")
        self.num_subdomains = num_subdomains
        self.owner = owner

    def composite(self, p, l):
        nr, ng = _i64(), _i64()
        _load().orc_composite_size(self._h, p, l, ctypes.byref(nr), ctypes.byref(ng))
        real = np.empty(nr.value, dtype=np.int32)
        ghost = np.empty(ng.value, dtype=np.int32)
        _load().orc_get_composite(self._h, p, l, _p(real), _p(ghost))
        return real, ghost

    # ---- solve ----
    def cycle(self, b, x, num_fac_cycles=2, relax_sweeps=1, subdomains=None, nthreads=1):
        """One AMG-DD cycle in place on x (only the listed subdomains update their owned dofs)."""
        lst = None if subdomains is None else np.ascontiguousarray(subdomains, dtype=np.int32)
        _load().orc_cycle(self._h, _p(b), _p(x), num_fac_cycles, relax_sweeps, _p(lst),
                          0 if lst is None else len(lst), nthreads)

    def residual_norm(self, b, x):
        return _load().orc_residual_norm(self._h, _p(b), _p(x))

    def solve(self, b, x, num_cycles, num_fac_cycles=2, relax_sweeps=1, nthreads=1):
        res = np.empty(num_cycles + 1, dtype=np.float64)
        _load().orc_solve(self._h, _p(b), _p(x), num_cycles, num_fac_cycles, relax_sweeps, _p(res), nthreads)
        return res

    def fac_local(self, p, r0, num_fac_cycles, relax_sweeps):
        real, ghost = self.composite(p, 0)
        out = np.empty(len(real) + len(ghost), dtype=np.float64)
        r0 = np.ascontiguousarray(r0, dtype=np.float64)
        _load().orc_fac_local(self._h, p, _p(r0), num_fac_cycles, relax_sweeps, _p(out))
        return out

    def relax(self, l, u, f, mask=None, dinv=None, nsweeps=1):
        u = np.array(u, dtype=np.float64)
        f = np.ascontiguousarray(f, dtype=np.float64)
        m = None if mask is None else np.ascontiguousarray(mask, dtype=np.int8)
        d = None if dinv is None else np.ascontiguousarray(dinv, dtype=np.float64)
        _load().orc_relax(self._h, l, _p(u), _p(f), _p(m), _p(d), nsweeps)
        return u

    def vcycle(self, b, x, nu1=1, nu2=1):
        x = np.array(x, dtype=np.float64)
        _load().orc_vcycle(self._h, _p(np.ascontiguousarray(b, dtype=np.float64)), _p(x), nu1, nu2)
        return x

    def coarse_solve(self, rhs):
        x = np.array(rhs, dtype=np.float64)
        _load().orc_coarse_solve(self._h, _p(x))
        return x

    def counters(self):
        out = np.zeros(3, dtype=np.int64)
        _load().orc_counters(self._h, _p(out))
        return {"A": int(out[0]), "P": int(out[1]), "R": int(out[2])}

    def dropped(self):
        return int(_load().orc_dropped(self._h))

    def overhead(self, nthreads=1):
        return _load().orc_overhead(self._h, nthreads)


def max_threads():
    return int(_load().orc_max_threads())
