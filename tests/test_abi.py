"""C-ABI checks that need no GPU: the library loads, exports every symbol include/amgdd.h
declares, validates its arguments before touching the device, and refuses to compute without
a CUDA device (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "amgdd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(amgdd_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_1906_10575_b200 as m
    names = _declared_symbols()
    assert len(names) >= 15
    for name in names:
        assert hasattr(m.lib, name), f"libamgdd.so does not export {name}"
    assert set(names) == set(m.EXPORTS)


def test_binding_has_the_same_names():
    import paper_1906_10575_b200 as m
    for name in _declared_symbols():
        if name == "amgdd_last_error_detail":
            continue
        assert callable(getattr(m, name)), name


def test_strerror_covers_all_codes():
    import paper_1906_10575_b200 as m
    seen = set()
    for code in range(0, -10, -1):
        s = m.amgdd_strerror(code)
        assert s and s != "unknown status"
        seen.add(s)
    assert len(seen) == 10
    assert m.amgdd_strerror(-99) == "unknown status"


def _setup(m, p, **kw):
    args = dict(n=p.n, rowptr=p.rowptr, colind=p.colind, vals=p.vals, num_subdomains=p.num_subdomains,
                owner=p.owner, eta=p.eta, num_ghost=1, max_levels=25, theta=p.theta, coarse_max=p.coarse_max)
    args.update(kw)
    return m.amgdd_setup(**args)


def test_argument_validation_precedes_device_use():
    import paper_1906_10575_b200 as m
    p = wl.make_config(1, 9)
    bad = [
        (dict(n=0), -1), (dict(num_subdomains=0), -1), (dict(eta=-1), -1), (dict(num_ghost=0), -1),
        (dict(theta=0.0), -1), (dict(theta=1.5), -1), (dict(max_levels=0), -1), (dict(coarse_max=0), -1),
        (dict(rowptr=None), -1),
    ]
    for kw, code in bad:
        with pytest.raises(m.AmgddError) as e:
            _setup(m, p, **kw)
        assert e.value.code == code, kw
    # malformed CSR
    rp = p.rowptr.copy(); rp[0] = 1
    ci = p.colind.copy(); ci[1], ci[2] = ci[2], ci[1]           # row 0 columns no longer ascending? use row 1
    v_neg = p.vals.copy(); v_neg[p.rowptr[5]:p.rowptr[6]][p.colind[p.rowptr[5]:p.rowptr[6]] == 5] = -4.0
    ci_oob = p.colind.copy(); ci_oob[-1] = p.n
    # drop one off-diagonal entry -> structurally unsymmetric
    keep = np.ones(p.nnz, dtype=bool); keep[p.rowptr[0] + 1] = False
    rp_u = np.concatenate([[0], np.cumsum(np.add.reduceat(keep.astype(np.int64), p.rowptr[:-1]))])
    v_nan = p.vals.copy(); v_nan[p.rowptr[7] + 1] = np.nan         # a non-finite off-diagonal (the diagonal test alone misses it)
    v_inf = p.vals.copy(); v_inf[p.rowptr[3]] = -np.inf
    for kw in [dict(rowptr=rp), dict(colind=ci), dict(vals=v_neg), dict(colind=ci_oob), dict(vals=v_nan), dict(vals=v_inf),
               dict(rowptr=rp_u, colind=p.colind[keep], vals=p.vals[keep])]:
        with pytest.raises(m.AmgddError) as e:
            _setup(m, p, **kw)
        assert e.value.code == -2, list(kw)
    own = p.owner.copy(); own[0] = 7
    with pytest.raises(m.AmgddError) as e:
        _setup(m, p, owner=own)
    assert e.value.code == -3
    with pytest.raises(m.AmgddError) as e:
        _setup(m, p, num_subdomains=5)            # subdomain 4 owns nothing
    assert e.value.code == -3


def test_no_cpu_fallback():
    import torch
    import paper_1906_10575_b200 as m
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(m.AmgddError) as e:
        _setup(m, wl.make_config(1))
    assert e.value.code == -8 and "no CPU fallback" in str(e.value)


def test_product_does_not_import_the_oracle():
    # the CUDA path and the oracle share no code and neither imports the other
    pkg = os.path.join(ROOT, "paper_1906_10575_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert not re.search(r'#include\s+"[^"]*oracle', txt), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1906_10575_b200 import" not in txt and "import paper_1906_10575_b200" not in txt, f
            assert not re.search(r'#include\s+"[^"]*(csrc|amgdd\.h)', txt), f


def test_stats_struct_layout_matches_the_header(tmp_path):
    """The ctypes mirror of amgdd_stats_t / amgdd_way_t has the size and field offsets the C compiler gives the
    header's structs (a silent mismatch would corrupt memory in amgdd_get_stats)."""
    import shutil
    import subprocess
    import paper_1906_10575_b200 as m
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no C compiler")
    fields = [n for n, _ in m.AmgddStats._fields_]
    src = ['#include <stdio.h>', '#include <stddef.h>', '#include "amgdd.h"', 'int main(void) {',
           '  printf("%zu %zu\\n", sizeof(amgdd_stats_t), sizeof(amgdd_way_t));']
    src += [f'  printf("{n} %zu\\n", offsetof(amgdd_stats_t, {n}));' for n in fields]
    src += ['  return 0;', '}']
    c = tmp_path / "layout.c"
    c.write_text("\n".join(src))
    exe = tmp_path / "layout"
    subprocess.run([gcc, "-I", os.path.join(ROOT, "include"), str(c), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split("\n")
    size_stats, size_way = map(int, out[0].split())
    assert size_stats == ctypes.sizeof(m.AmgddStats)
    assert size_way == m.WAY_DTYPE.itemsize
    for line in out[1:]:
        if line:
            name, off = line.split()
            assert getattr(m.AmgddStats, name).offset == int(off), name
