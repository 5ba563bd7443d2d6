"""Seeded synthetic inputs for AMG-DD.

This module is the ONE thing the oracle tests and the CUDA-path tests share.  It only makes
inputs (matrices in CSR, owner arrays, right-hand sides); none of the method's arithmetic
(strength, coarsening, interpolation, relaxation ...) lives here.

Conventions:
  * dof index i = x + nx*(y + ny*z), x fastest; Dirichlet boundary eliminated (interior unknowns
    only, boundary-adjacent rows are shorter); no h^2 scaling.
  * CSR with int64 rowptr, int32 colind strictly ascending per row, float64 vals.
  * block owner per dimension floor(c*parts/n), p = bx + px*(by + py*bz).
  * RNG: std::mt19937_64(seed), u = (draw >> 11) * 2^-53 in index order; b_i = 2u - 1.

The five BASELINE.json configs stand in for the paper's MFEM/METIS problems (PAPER.md line 261,
Problems 1 and 2), which are not available in this container.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libwl_mt64.so")
_SRC = os.path.join(_HERE, "mt64.cpp")


def build(force: bool = False) -> str:
    """Compile the tiny mt19937_64 helper with g++ (seconds)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", _SO])
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.wl_uniform.argtypes = [ctypes.c_uint64, ctypes.c_int64, ctypes.c_void_p]
        _lib.wl_raw.argtypes = [ctypes.c_uint64, ctypes.c_int64, ctypes.c_void_p]
    return _lib


def uniform(seed: int, n: int) -> np.ndarray:
    """n uniforms in [0,1) from std::mt19937_64(seed): (draw >> 11) * 2^-53."""
    out = np.empty(n, dtype=np.float64)
    _load().wl_uniform(seed, n, out.ctypes.data)
    return out


def raw_draws(seed: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.uint64)
    _load().wl_raw(seed, n, out.ctypes.data)
    return out


def rhs(seed: int, n: int) -> np.ndarray:
    """b_i = 2u_i - 1, b ~ U(-1,1) (BASELINE.json configs)."""
    return 2.0 * uniform(seed, n) - 1.0


# --------------------------------------------------------------------------------------------
# structured-grid CSR assembly
# --------------------------------------------------------------------------------------------
def _coords(shape):
    """x, y(, z) coordinate arrays of every dof, flattened in dof order (x fastest)."""
    grids = np.meshgrid(*[np.arange(s, dtype=np.int64) for s in shape[::-1]], indexing="ij")
    return [g.ravel() for g in grids[::-1]]


def _assemble(shape, offsets, values_fn):
    """CSR from a list of stencil offsets (each a tuple in x,y(,z)); offsets must be given in
    ascending linear-offset order so that columns come out strictly ascending.
    values_fn(k, valid_mask) -> array of the coefficient of offset k at every dof."""
    dims = len(shape)
    N = int(np.prod(shape))
    c = _coords(shape)
    strides = [1]
    for d in range(dims - 1):
        strides.append(strides[-1] * shape[d])
    lin = [sum(o[d] * strides[d] for d in range(dims)) for o in offsets]
    assert all(lin[i] < lin[i + 1] for i in range(len(lin) - 1)), "offsets not ascending"
    K = len(offsets)
    mask = np.empty((N, K), dtype=bool)
    cols = np.empty((N, K), dtype=np.int32)
    vals = np.empty((N, K), dtype=np.float64)
    idx = np.arange(N, dtype=np.int64)
    for k, o in enumerate(offsets):
        ok = np.ones(N, dtype=bool)
        for d in range(dims):
            if o[d] != 0:
                cc = c[d] + o[d]
                ok &= (cc >= 0) & (cc < shape[d])
        mask[:, k] = ok
        cols[:, k] = (idx + lin[k]).astype(np.int32)
        vals[:, k] = values_fn(k, ok)
    rowptr = np.zeros(N + 1, dtype=np.int64)
    np.cumsum(mask.sum(axis=1), out=rowptr[1:])
    return rowptr, np.ascontiguousarray(cols[mask]), np.ascontiguousarray(vals[mask])


def poisson2d_5pt(n):
    """2D 5-point: diag 4, neighbours -1, n x n interior grid (config 1)."""
    offs = [(0, -1), (-1, 0), (0, 0), (1, 0), (0, 1)]
    v = [-1.0, -1.0, 4.0, -1.0, -1.0]
    return _assemble((n, n), offs, lambda k, ok: np.full(ok.shape, v[k]))


def poisson3d_7pt(n):
    """3D 7-point: diag 6, neighbours -1, n^3 interior grid (config 2)."""
    offs = [(0, 0, -1), (0, -1, 0), (-1, 0, 0), (0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)]
    v = [-1.0, -1.0, -1.0, 6.0, -1.0, -1.0, -1.0]
    return _assemble((n, n, n), offs, lambda k, ok: np.full(ok.shape, v[k]))


def fe27_3d(n):
    """3D 27-point trilinear-FE Laplacian on a uniform hex mesh: centre 8/3, face 0.0 (STORED),
    edge -1/6, corner -1/12 (config 3; stands in for Problem 1's linear FE)."""
    offs, v = [], []
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                offs.append((dx, dy, dz))
                v.append({0: 8.0 / 3.0, 1: 0.0, 2: -1.0 / 6.0, 3: -1.0 / 12.0}[abs(dx) + abs(dy) + abs(dz)])
    return _assemble((n, n, n), offs, lambda k, ok: np.full(ok.shape, v[k]))


def _fv_diffusion(shape, kcell, axis_scale):
    """Cell-centred FV of -div(k grad u): interior face T = 2 ka kb/(ka+kb) (harmonic mean),
    boundary face T = 2 kc (Dirichlet), a_ii = sum T, a_ij = -T; faces along axis d scaled by
    axis_scale[d]."""
    dims = len(shape)
    c = _coords(shape)
    strides = [1]
    for d in range(dims - 1):
        strides.append(strides[-1] * shape[d])
    N = int(np.prod(shape))
    idx = np.arange(N, dtype=np.int64)
    # face transmissibilities toward -d and +d for every cell
    T = {}
    for d in range(dims):
        for sgn in (-1, 1):
            cc = c[d] + sgn
            inside = (cc >= 0) & (cc < shape[d])
            nb = np.where(inside, idx + sgn * strides[d], idx)
            kb = kcell[nb]
            t = np.where(inside, 2.0 * kcell * kb / (kcell + kb), 2.0 * kcell) * axis_scale[d]
            T[(d, sgn)] = t
    # diagonal: sum faces in a fixed order (-x,+x,-y,+y,-z,+z)
    diag = np.zeros(N)
    for d in range(dims):
        for sgn in (-1, 1):
            diag = diag + T[(d, sgn)]
    offs = []
    for d in reversed(range(dims)):
        o = [0] * dims
        o[d] = -1
        offs.append(tuple(o))
    offs.append(tuple([0] * dims))
    for d in range(dims):
        o = [0] * dims
        o[d] = 1
        offs.append(tuple(o))

    def val(k, ok):
        o = offs[k]
        if all(x == 0 for x in o):
            return diag
        d = [i for i in range(dims) if o[i] != 0][0]
        return -T[(d, o[d])]

    return _assemble(shape, offs, val)


def varcoef3d_7pt(n, seed):
    """Config 4: k_c = exp(g_c), g_c ~ N(0,1) by Box-Muller on the seed stream in index order,
    g = sqrt(-2 ln(1-u1)) cos(2 pi u2), one value per pair of draws."""
    N = n ** 3
    u = uniform(seed, 2 * N)
    g = np.sqrt(-2.0 * np.log(1.0 - u[0::2])) * np.cos(2.0 * np.pi * u[1::2])
    return _fv_diffusion((n, n, n), np.exp(g), (1.0, 1.0, 1.0))


def aniso2d_jumps(n, seed, eps=1e-3, blocks=16, hi=1e4):
    """Config 5: -dx(k dx u) - eps dy(k dy u); k constant on (n/blocks)^2 blocks, 1 or `hi` by the
    top bit of one seed draw per block in row-major block order."""
    bits = (raw_draws(seed, blocks * blocks) >> np.uint64(63)).astype(np.int64).reshape(blocks, blocks)
    kb = np.where(bits == 1, hi, 1.0)
    x, y = _coords((n, n))
    kcell = kb[y * blocks // n, x * blocks // n]
    return _fv_diffusion((n, n), kcell, (1.0, eps))


def rotated_aniso2d_9pt(n, theta=3.0 * np.pi / 16.0, eps=1e-3):
    """Problem 2 of the paper (eq. 33): -div(K grad u), K = Q^T D Q with the rotation angle theta and
    D = diag(1, eps), discretised with bilinear finite elements on a uniform n x n interior grid (Dirichlet
    boundary eliminated, no h scaling).  With K = [[a, b], [b, d]] the 9-point row is: centre 4(a+d)/3, (+-1, 0)
    (d-2a)/3, (0, +-1) (a-2d)/3, (+1,+1) and (-1,-1) -(a+d)/6 - b/2, (+1,-1) and (-1,+1) -(a+d)/6 + b/2: some
    off-diagonals are positive (reading A11 of DESIGN.md)."""
    c, s_ = np.cos(theta), np.sin(theta)
    a, b, d = c * c + eps * s_ * s_, (1.0 - eps) * c * s_, s_ * s_ + eps * c * c
    offs, v = [], []
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            offs.append((dx, dy))
            if dx == 0 and dy == 0:
                v.append(4.0 * (a + d) / 3.0)
            elif dy == 0:
                v.append((d - 2.0 * a) / 3.0)
            elif dx == 0:
                v.append((a - 2.0 * d) / 3.0)
            else:
                v.append(-(a + d) / 6.0 - (b / 2.0 if dx * dy > 0 else -b / 2.0))
    return _assemble((n, n), offs, lambda k, ok: np.full(ok.shape, v[k]))


def block_owner(shape, parts):
    """owner[i] for regular block partitions: per dimension floor(c*parts/n)."""
    c = _coords(shape)
    own = np.zeros(c[0].shape, dtype=np.int64)
    mul = 1
    for d in range(len(shape)):
        own += (c[d] * parts[d] // shape[d]) * mul
        mul *= parts[d]
    return own.astype(np.int32)


# --------------------------------------------------------------------------------------------
# the BASELINE.json configs (and scaled-down versions of the same recipe)
# --------------------------------------------------------------------------------------------
@dataclass
class Problem:
    name: str
    n: int
    rowptr: np.ndarray
    colind: np.ndarray
    vals: np.ndarray
    owner: np.ndarray
    num_subdomains: int
    b: np.ndarray
    eta: int
    theta: float
    coarse_max: int
    num_cycles: int
    num_fac_cycles: int = 2
    relax_sweeps: int = 1
    num_ghost: int = 1
    max_levels: int = 25
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self):
        return int(self.rowptr[-1])


def make_config(cfg: int, scale: int | None = None, eta: int | None = None, parts_per_dim: int | None = None) -> Problem:
    """BASELINE.json configs 1..5 (and 6: the paper's Problem 2, an extra workload).  `scale` overrides the grid edge (and keeps the subdomain block
    edge of the full config where it divides) to get smaller instances of the same recipe."""
    if cfg == 1:
        n = scale or 33
        rp, ci, v = poisson2d_5pt(n)
        pp = parts_per_dim or 2
        parts = (pp, pp)
        own = block_owner((n, n), parts)
        return Problem(f"cfg1-poisson2d-{n}", n * n, rp, ci, v, own, pp * pp, rhs(0, n * n),
                       eta if eta is not None else 1, 0.25, 16, 3, meta={"shape": (n, n), "parts": parts})
    if cfg == 2:
        n = scale or 64
        rp, ci, v = poisson3d_7pt(n)
        pp = parts_per_dim or max(1, n // 16)
        parts = (pp, pp, pp)
        own = block_owner((n, n, n), parts)
        return Problem(f"cfg2-poisson3d-{n}", n ** 3, rp, ci, v, own, pp ** 3, rhs(1, n ** 3),
                       eta if eta is not None else 2, 0.5, 64, 10, meta={"shape": (n,) * 3, "parts": parts})
    if cfg == 3:
        n = scale or 128
        rp, ci, v = fe27_3d(n)
        pp = parts_per_dim or max(1, n // 16)
        parts = (pp, pp, pp)
        own = block_owner((n, n, n), parts)
        return Problem(f"cfg3-fe27-{n}", n ** 3, rp, ci, v, own, pp ** 3, rhs(2, n ** 3),
                       eta if eta is not None else 1, 0.5, 64, 10, meta={"shape": (n,) * 3, "parts": parts})
    if cfg == 4:
        n = scale or 192
        rp, ci, v = varcoef3d_7pt(n, 3)
        pp = parts_per_dim or max(1, n // 12)
        parts = (pp, pp, pp)
        own = block_owner((n, n, n), parts)
        return Problem(f"cfg4-varcoef3d-{n}", n ** 3, rp, ci, v, own, pp ** 3, rhs(3 + 1000, n ** 3),
                       eta if eta is not None else 2, 0.5, 64, 10, meta={"shape": (n,) * 3, "parts": parts})
    if cfg == 5:
        n = scale or 2048
        rp, ci, v = aniso2d_jumps(n, 4)
        pp = parts_per_dim or max(1, n // 64)
        parts = (pp, pp)
        own = block_owner((n, n), parts)
        return Problem(f"cfg5-aniso2d-{n}", n * n, rp, ci, v, own, pp * pp, rhs(4 + 1000, n * n),
                       eta if eta is not None else 3, 0.25, 64, 15, meta={"shape": (n, n), "parts": parts})
    if cfg == 6:
        # not a BASELINE.json config: the paper's Problem 2 proper (rotated anisotropic diffusion),
        # SURVEY.md section 8(f) NEXT 3; 1024^2, 16 x 16 subdomains of 64^2, padding 1 as in the paper's GPU runs
        n = scale or 1024
        rp, ci, v = rotated_aniso2d_9pt(n)
        pp = parts_per_dim or max(1, n // 64)
        parts = (pp, pp)
        own = block_owner((n, n), parts)
        return Problem(f"cfg6-rotaniso2d-{n}", n * n, rp, ci, v, own, pp * pp, rhs(5 + 1000, n * n),
                       eta if eta is not None else 1, 0.25, 64, 10, meta={"shape": (n, n), "parts": parts})
    raise ValueError(f"unknown config {cfg}")


def poisson1d(n):
    """tridiag(-1, 2, -1), used by the closed-form pins."""
    offs = [(-1,), (0,), (1,)]
    v = [-1.0, 2.0, -1.0]
    return _assemble((n,), offs, lambda k, ok: np.full(ok.shape, v[k]))


def pivoting_band_matrix(n=24, seed=31):
    """A test input for the dense coarse solve (Alg. 4): a symmetric-PATTERN pentadiagonal matrix with a tiny
    positive diagonal and O(1) off-diagonals, so that Gaussian elimination with partial pivoting exchanges rows in
    (almost) every column.  Returns (rowptr int64, colind int32, vals, dense array)."""
    u = uniform(seed, 5 * n)
    rowptr, colind, vals = [0], [], []
    dense = np.zeros((n, n))
    k = 0
    for i in range(n):
        for j in range(max(0, i - 2), min(n, i + 3)):
            a = 1e-3 * (1.0 + u[k]) if i == j else (0.5 + u[k]) * (1.0 if (i + j) % 3 else -1.0)
            colind.append(j); vals.append(a); dense[i, j] = a
            k += 1
        rowptr.append(len(colind))
    return np.array(rowptr, dtype=np.int64), np.array(colind, dtype=np.int32), np.array(vals), dense
