"""NEXT 3 of SURVEY.md section 8(f) (paper P:335: renumbering the columns of the composite A_l is the dominant
setup cost, and no setup routine of the paper runs on the GPU): the composite-grid matrices are cut out of the
global level matrices, renumbered and packed on the device (csrc/amgdd_assemble.cu).  Index work only, so the
bar is bit-exactness: every array of every private (subdomain, level) block must be byte-identical to what the
host assembly writes (AMGDD_ASSEMBLE=host: CompositeBuilder + the host packer, which tests/test_pack_stream.py
decodes back to CSR and every parity test has exercised), and the solves on the two handles must agree to the bit.
The device assembly is the default path, so all other GPU tests compare it with the oracle as well."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

ARRAYS = ("gid", "dinv", "A", "P", "R")


def setup(p, monkeypatch, host):
    import paper_1906_10575_b200 as m
    if host:
        monkeypatch.setenv("AMGDD_ASSEMBLE", "host")
    else:
        monkeypatch.delenv("AMGDD_ASSEMBLE", raising=False)
    h = m.amgdd_setup(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.num_ghost, p.max_levels,
                      p.theta, p.coarse_max)
    assert m.amgdd_get_stats(h)["assembled_on_device"] == (0 if host else 1)
    return m, h


def compare_blocks(m, hd, hh, p, subdomains):
    nl = m.amgdd_num_levels(hd)
    private = 0
    for q in subdomains:
        a = m.amgdd_debug_read_block(hd, int(q), 0, "owned")
        b = m.amgdd_debug_read_block(hh, int(q), 0, "owned")
        assert a.size == 4 * int((p.owner == q).sum()) and np.array_equal(a, b), f"owned-dof list of subdomain {q}"
        for l in range(nl):
            for w in ARRAYS:
                a = m.amgdd_debug_read_block(hd, int(q), l, w)
                b = m.amgdd_debug_read_block(hh, int(q), l, w)
                assert a.size == b.size, f"size of {w}, subdomain {q}, level {l}: device {a.size}, host {b.size}"
                if a.size and not np.array_equal(a, b):
                    first = int(np.flatnonzero(a != b)[0])
                    raise AssertionError(f"{w} of subdomain {q}, level {l} differs from byte {first} of {a.size}")
                private += (w == "A" and a.size > 0)
    return private


def compare_solves(m, hd, hh, p, cycles):
    import torch
    out = []
    for h in (hd, hh):
        b = torch.from_numpy(p.b).cuda()
        x = torch.zeros(p.n, dtype=torch.float64, device="cuda")
        res = m.amgdd_solve(h, b, x, cycles, 2, 1)
        out.append((np.asarray(res), x.cpu().numpy()))
    assert np.array_equal(out[0][0], out[1][0]), "residual norms of the two assemblies differ"
    assert np.array_equal(out[0][1], out[1][1]), "iterates of the two assemblies differ"


@pytest.mark.parametrize("cfg,scale,kw", [
    (1, None, {}),                                  # 4 subdomains, coarse levels shared
    (2, 32, {}),                                    # 3D 7-point, eta 2
    (3, 32, {"eta": 2}),                            # 27-point: long rows, several groups per slice
    (4, 48, {}),                                    # variable coefficients: irregular coarsening, ragged rows
    (5, 256, {}),                                   # 2D anisotropic, eta 3
    (6, 192, {"eta": 2, "parts_per_dim": 4}),       # rotated anisotropy, 9-point
])
def test_device_assembly_is_byte_identical(cfg, scale, kw, monkeypatch):
    p = wl.make_config(cfg, scale, **kw)
    m, hd = setup(p, monkeypatch, host=False)
    m, hh = setup(p, monkeypatch, host=True)
    sd, sh = m.amgdd_get_stats(hd), m.amgdd_get_stats(hh)
    for k in ("nnz_composite_real", "sum_real", "sum_ghost", "shared_level_instances", "stream_bytes_fac_iter",
              "model_bytes_fac_iter", "max_n_bar"):
        assert sd[k] == sh[k], k
    rng = np.random.default_rng(cfg)
    P = p.num_subdomains
    subs = np.arange(P) if P <= 64 else np.unique(np.concatenate([[0, P - 1], rng.choice(P, 40, replace=False)]))
    assert compare_blocks(m, hd, hh, p, subs) > 0, "no private level was compared"
    compare_solves(m, hd, hh, p, 2)
    m.amgdd_destroy(hd)
    m.amgdd_destroy(hh)


def test_wide_streams_and_small_batches(monkeypatch):
    # 2 x 2 subdomains of a 600 x 600 grid: |D-bar_0| > 90000 > 65535, so the private level-0 streams carry
    # 32-bit column indices; batches of one subdomain exercise the re-use of the batch buffers
    monkeypatch.setenv("AMGDD_SETUP_BATCH", "1")
    p = wl.make_config(1, 600, parts_per_dim=2)
    m, hd = setup(p, monkeypatch, host=False)
    m, hh = setup(p, monkeypatch, host=True)
    assert m.amgdd_get_stats(hd)["max_n_bar"] > 65536
    assert compare_blocks(m, hd, hh, p, np.arange(p.num_subdomains)) > 0
    compare_solves(m, hd, hh, p, 1)
    m.amgdd_destroy(hd); m.amgdd_destroy(hh)
    p = wl.make_config(2, 32)
    m, hd = setup(p, monkeypatch, host=False)
    m, hh = setup(p, monkeypatch, host=True)
    assert compare_blocks(m, hd, hh, p, np.arange(p.num_subdomains)) > 0
    m.amgdd_destroy(hd); m.amgdd_destroy(hh)


@pytest.mark.parametrize("window", ["32", "1024"])
def test_other_sort_windows(window, monkeypatch):
    monkeypatch.setenv("AMGDD_WINDOW", window)
    p = wl.make_config(4, 24)
    m, hd = setup(p, monkeypatch, host=False)
    m, hh = setup(p, monkeypatch, host=True)
    assert compare_blocks(m, hd, hh, p, np.arange(p.num_subdomains)) > 0
    compare_solves(m, hd, hh, p, 1)
    m.amgdd_destroy(hd); m.amgdd_destroy(hh)


def test_large_window_falls_back_to_the_host_packer(monkeypatch):
    # the device sort ranks the rows of a window inside one shared-memory tile of 1024 rows
    monkeypatch.setenv("AMGDD_WINDOW", "2048")
    p = wl.make_config(2, 32)
    import paper_1906_10575_b200 as m
    h = m.amgdd_setup(p.n, p.rowptr, p.colind, p.vals, p.num_subdomains, p.owner, p.eta, p.num_ghost, p.max_levels,
                      p.theta, p.coarse_max)
    assert m.amgdd_get_stats(h)["assembled_on_device"] == 0
    m.amgdd_destroy(h)


def test_index_sets_on_the_device_and_on_the_host(monkeypatch):
    """The rest of NEXT 3: D_l^p and the ghost layers grown on the device (bitmaps, one CTA per subdomain) against the host's
    breadth-first search (AMGDD_INDEX_SETS=host), byte for byte; a frontier that does not fit the device scratch hands the
    batch to the host."""
    import paper_1906_10575_b200 as m
    for cfg, scale, kw in ((4, 48, {}), (5, 256, {}), (3, 32, {"eta": 4}), (1, 37, {"parts_per_dim": 3, "eta": 0})):
        p = wl.make_config(cfg, scale, **kw)
        monkeypatch.delenv("AMGDD_INDEX_SETS", raising=False)
        try:
            _, hd = setup(p, monkeypatch, host=False)
        except m.AmgddError as e:                       # eta = 0 may leave interpolation stencils outside the grid (A7): both paths refuse
            assert e.code == -6
            monkeypatch.setenv("AMGDD_INDEX_SETS", "host")
            with pytest.raises(m.AmgddError):
                setup(p, monkeypatch, host=False)
            continue
        assert m.amgdd_get_stats(hd)["index_sets_on_device"] == 1
        monkeypatch.setenv("AMGDD_INDEX_SETS", "host")
        _, hs = setup(p, monkeypatch, host=False)
        assert m.amgdd_get_stats(hs)["index_sets_on_device"] == 0
        assert compare_blocks(m, hd, hs, p, np.arange(p.num_subdomains)) > 0
        sd, sh = m.amgdd_get_stats(hd), m.amgdd_get_stats(hs)
        for k in ("nnz_composite_real", "sum_real", "sum_ghost", "shared_level_instances", "stream_bytes_fac_iter", "overhead"):
            assert sd[k] == sh[k], k
        m.amgdd_destroy(hd); m.amgdd_destroy(hs)
    # one subdomain that owns 640 x 640 dofs: more seeds than the frontier scratch holds
    monkeypatch.delenv("AMGDD_INDEX_SETS", raising=False)
    p = wl.make_config(1, 640, parts_per_dim=1)
    _, h = setup(p, monkeypatch, host=False)
    assert m.amgdd_get_stats(h)["index_sets_on_device"] == 0
    import torch
    b = torch.from_numpy(p.b).cuda()
    x = torch.zeros(p.n, dtype=torch.float64, device="cuda")
    res = m.amgdd_solve(h, b, x, 2)
    assert res[2] < res[1] < res[0]
    m.amgdd_destroy(h)
