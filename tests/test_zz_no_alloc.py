"""amgdd_residual_norm_static: the residual norm for callers that cannot allocate device memory.

Some users of this library need || b - A x ||_2 at a place where cudaMalloc is not an option: their own
memory pool (or a framework's caching allocator) already holds the GPU's memory, they have no
amgdd_handle_t (amgdd_setup allocates the whole hierarchy), or they sit in a loop that must not meet the
device-wide synchronisation of cudaFree.  For them the library has ONE entry point that allocates nothing:
its scratch (a partial sum per 256 rows and an arrival counter) is a fixed device array inside
libamgdd.so, shared by every call on that GPU, hence the row limit AMGDD_STATIC_MAX_ROWS.

What is checked: the norm against the existing, handle-based amgdd_residual_norm (same bar as the parity
tests, 1e-10 relative), on calls that follow each other with different vectors and a different, smaller
matrix in between -- the shared array keeps what the previous call wrote, and nothing of it may leak into
the next result.  This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It also has to pass alone in a fresh process, where its first call
is the one that looks up the array's device address.
"""
import ctypes

import numpy as np
import pytest

import workloads as wl

RTOL = 1e-10     # the bar of tests/test_gpu_parity.py


def _device_csr(torch, p):
    return (torch.from_numpy(p.rowptr.astype(np.int64)).cuda(), torch.from_numpy(p.colind.astype(np.int32)).cuda(),
            torch.from_numpy(p.vals.astype(np.float64)).cuda())


@pytest.mark.gpu
def test_static_residual_norm_matches_the_handle_path_on_consecutive_calls():
    import torch
    import paper_1906_10575_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    big = wl.make_config(4, 48)          # 48^3 variable-coefficient diffusion: 110592 rows = 432 CTAs, several waves of partial sums
    small = wl.make_config(1)            # 33 x 33 Poisson: 1089 rows = 4 full CTAs and a ragged one
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    rng = np.random.default_rng(20241106)
    cases = []
    for p in (big, small):
        h = m.amgdd_setup(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, 1, p.max_levels, p.theta, p.coarse_max)
        cases.append((p, h, _device_csr(torch, p), torch.from_numpy(p.b).cuda(), torch.empty(p.n, dtype=torch.float64, device="cuda")))
    # big, big again with another x, small (fewer CTAs than the call before: stale partial sums lie behind its own), big, small
    for k, which in enumerate((0, 0, 1, 0, 1)):
        p, h, (rp, ci, v), b, r = cases[which]
        x = torch.from_numpy(rng.uniform(-1.0, 1.0, p.n) * 10.0 ** k).cuda()
        want = m.amgdd_residual_norm(h, b, x)                      # existing path: scratch owned by the handle
        out.fill_(float("nan"))
        r.fill_(float("nan"))
        m.amgdd_residual_norm_static(p.n, rp, ci, v, b, x, out, r=r)
        torch.cuda.synchronize()
        got = float(out.item())
        assert want > 0.0 and abs(got - want) <= RTOL * want, (k, which, got, want)
        # the residual vector it leaves is the one whose norm it reports
        rn = float(torch.linalg.vector_norm(r).item())
        assert abs(rn - want) <= RTOL * want, (k, which, rn, want)
        # and r = NULL changes nothing
        out.fill_(float("nan"))
        m.amgdd_residual_norm_static(p.n, rp, ci, v, b, x, out)
        torch.cuda.synchronize()
        assert float(out.item()) == got, (k, which)
    # beyond the fixed array: refused with the limit in the message, nothing launched, the output untouched
    p, h, (rp, ci, v), b, r = cases[0]
    out.fill_(-1.0)
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_residual_norm_static(m.STATIC_MAX_ROWS + 1, rp, ci, v, b, b, out)
    assert e.value.code == -1 and "AMGDD_STATIC_MAX_ROWS" in str(e.value) and str(m.STATIC_MAX_ROWS) in str(e.value)
    torch.cuda.synchronize()
    assert float(out.item()) == -1.0
    for _, h, *_ in cases:
        m.amgdd_destroy(h)


def test_static_residual_norm_checks_its_arguments_before_the_device():
    """Needs no GPU: the size limit and null pointers are reported before any CUDA call."""
    import paper_1906_10575_b200 as m
    dummy = ctypes.c_double(0.0)
    a = ctypes.addressof(dummy)
    assert m.lib.amgdd_residual_norm_static(m.STATIC_MAX_ROWS + 1, a, a, a, a, a, None, a, None) == -1
    assert b"AMGDD_STATIC_MAX_ROWS" in m.lib.amgdd_last_error_detail()
    assert m.lib.amgdd_residual_norm_static(0, a, a, a, a, a, None, a, None) == -1
    assert m.lib.amgdd_residual_norm_static(8, a, a, a, a, a, None, None, None) == -1
    # the header's constant and the binding's agree
    import os
    import re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "amgdd.h")).read()
    assert int(re.search(r"#define AMGDD_STATIC_MAX_ROWS (\d+)", hdr).group(1)) == m.STATIC_MAX_ROWS
