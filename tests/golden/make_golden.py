"""Writes the stored expected values under tests/golden/.  Calls ONLY oracle/ (and the seeded input
generators of workloads/): no value here ever comes from the CUDA path.

The paper (arXiv 1906.10575) prints no worked numerical example for the AlgFAC path (its results are
figures), so there is no fixture "from the paper"; the pins of the oracle are closed forms, brute force
and independent formulations (tests/test_oracle_pins.py).  These files are regression anchors of the
pinned oracle: residual norms per AMG-DD cycle of BASELINE.json configs[0] (full size) and of a small
instance of configs[3], 17 significant digits.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402
from oracle import Oracle  # noqa: E402

CASES = [("config1_resnorms.txt", 1, None, 0), ("config4_scale24_resnorms.txt", 4, 24, 0),
         ("config1_cfjacobi_resnorms.txt", 1, None, 1)]


def resnorms(cfg, scale, smoother):
    p = wl.make_config(cfg, scale)
    o = Oracle(p.n, p.rowptr, p.colind, p.vals, p.theta, p.max_levels, p.coarse_max)
    o.set_partition(p.num_subdomains, p.owner, p.eta, p.num_ghost)
    o.set_smoother(smoother)
    x = np.zeros(p.n)
    return p, o.solve(p.b, x, p.num_cycles, p.num_fac_cycles, p.relax_sweeps)


if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    for name, cfg, scale, smoother in CASES:
        p, res = resnorms(cfg, scale, smoother)
        with open(os.path.join(here, name), "w") as f:
            f.write(f"# ||b - A x_k||_2, k = 0..{p.num_cycles}: {p.name}, P = {p.num_subdomains}, eta = {p.eta}, "
                    f"{p.num_fac_cycles} AlgFAC V({p.relax_sweeps},{p.relax_sweeps}) cycles per AMG-DD cycle "
                    f"(Alg. 2 P:468-480, Alg. 4 P:499-521), smoother {smoother}; written by tests/golden/make_golden.py from oracle/ only\n")
            for r in res:
                f.write(f"{r:.17e}\n")
        print(name, res)
