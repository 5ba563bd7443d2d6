"""Build libamgdd.so (hand-written sm_100a CUDA + host setup) in-tree with nvcc."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["amgdd_api.cu", "amgdd_kernels.cu", "amgdd_fac.cu", "amgdd_assemble.cu", "amgdd_static.cu", "amgdd_hierarchy.cpp", "amgdd_composite.cpp", "amgdd_pack.cpp", "amgdd_shard.cpp"]
HEADERS = ["amgdd_host.hpp", "amgdd_kernels.cuh", "amgdd_assemble.cuh", "amgdd_stream.hpp", os.path.join("..", "..", "include", "amgdd.h")]
LIB = os.path.join(HERE, "libamgdd.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--extended-lambda", "-Xcompiler", "-fPIC,-O3,-pthread", "-shared",
]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("AMGDD_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + \
          [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libamgdd.so")
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
