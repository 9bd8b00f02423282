"""Build libhydro_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1604_03360_b200.build [--force]

The library is the product: there is no CPU fallback, and ``binding`` raises if it is missing.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhydro_b200.so")
PROBE_LIB = os.path.join(HERE, "libbench_probe.so")   # bench.py's FMA-rate probe: a measurement helper, not the product
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-diag-suppress", "221", "-shared", "-Xcompiler", "-fPIC"]


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh"))) + \
        [os.path.join(os.path.dirname(HERE), "include", "hydro.h")]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        tmp = LIB + ".tmp%d" % os.getpid()
        cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              [os.path.join(CSRC, "hydro.cu"), "-o", tmp, "-lcuda"]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    psrc = os.path.join(CSRC, "bench_probe.cu")
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(psrc) > os.path.getmtime(PROBE_LIB):
        tmp = PROBE_LIB + ".tmp%d" % os.getpid()
        subprocess.check_call([NVCC] + FLAGS + [psrc, "-o", tmp])
        os.replace(tmp, PROBE_LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
