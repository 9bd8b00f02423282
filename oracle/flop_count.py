"""TEST INFRASTRUCTURE.  Builds and runs oracle/flop_count.cpp (the oracle's formulas on a counting scalar
type) and returns the operation counts as a dict.  `python -m oracle.flop_count` prints them and rewrites
tests/golden/flop_counts.txt."""
from __future__ import annotations

import os
import subprocess
import tempfile

_HERE = os.path.dirname(os.path.abspath(__file__))


def counts() -> dict:
    exe = os.path.join(tempfile.gettempdir(), "hydro_flop_count_%d" % os.getpid())
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-w", os.path.join(_HERE, "flop_count.cpp"), "-o", exe])
    try:
        out = subprocess.check_output([exe], text=True)
    finally:
        os.remove(exe)
    return {k: int(v) for k, v in (line.split() for line in out.strip().splitlines())}


if __name__ == "__main__":
    c = counts()
    path = os.path.join(os.path.dirname(_HERE), "tests", "golden", "flop_counts.txt")
    with open(path, "w") as fh:
        fh.write("# Floating-point operations of the oracle's formulas as literally written (oracle/flop_count.cpp:\n"
                 "# add, sub, mul, div, sqrt, abs, max, min = 1 each), assembled per cell of one L(u) and of one RK3\n"
                 "# step.  Written by `python -m oracle.flop_count`; calls only oracle/.\n"
                 "# The roofline numerator of bench.py is SURVEY.md 8(d)'s smaller textbook count with shared\n"
                 "# subexpressions (2327 / 4757 / 1257 per L(u)); these literal counts are its upper companion.\n")
        for k, v in c.items():
            fh.write("%s %d\n" % (k, v))
            print(k, v)
