"""Build the oracle's C library (test infrastructure; see nko.h).

  libnko.so      gcc -O2 -ffp-contract=off -fopenmp          the oracle
  libnko_fma.so  same source, -mfma -ffp-contract=fast        used only to measure the oracle's own
                                                              rounding band
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nko.c")
HDR = os.path.join(HERE, "nko.h")
LIB = os.path.join(HERE, "libnko.so")
LIB_FMA = os.path.join(HERE, "libnko_fma.so")

COMMON = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
          "-fno-fast-math", SRC, "-lm"]


def _stale(lib: str) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(s) > t for s in (SRC, HDR, os.path.abspath(__file__)))


def cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            return " fma " in f.read().replace("\n", " ")
    except OSError:
        return False


def build(force: bool = False, verbose: bool = False) -> str:
    jobs = [(LIB, ["-ffp-contract=off", "-o", LIB]),
            (LIB_FMA, ["-mfma", "-ffp-contract=fast", "-o", LIB_FMA])]
    for lib, extra in jobs:
        if force or _stale(lib):
            cmd = COMMON + extra
            if verbose:
                print(" ".join(cmd), file=sys.stderr)
            subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
