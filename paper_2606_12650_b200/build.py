"""Build libnk.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_12650_b200.build [--force] [--verbose]

Objects are compiled in parallel (one nvcc per translation unit) into csrc/build/, then linked
into paper_2606_12650_b200/libnk.so.  The .so is git-ignored but travels to the GPU box.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libnk.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

SOURCES = ["nk_api.cu", "nk_setup.cu", "nk_ax_tma.cu", "nk_gs.cu", "nk_vec.cu", "nk_geom.cu", "nk_dist.cu", "nk_probe.cu", "nk_basis.cpp"]
HEADERS = ["nk_internal.h", "nk_host.h", "nk_reduce.cuh"]

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-Xcompiler", "-fopenmp",
         "-Xptxas", "-v"]
EXTRA = os.environ.get("NK_NVCC_EXTRA", "").split()


def _newest_header() -> float:
    paths = [os.path.join(CSRC, h) for h in HEADERS] + [os.path.join(INCLUDE, "nk.h"), os.path.abspath(__file__)]
    return max(os.path.getmtime(p) for p in paths)


def _compile(src: str, force: bool, verbose: bool):
    obj = os.path.join(OBJDIR, os.path.splitext(src)[0] + ".o")
    path = os.path.join(CSRC, src)
    if (not force and os.path.exists(obj) and os.path.getmtime(obj) > os.path.getmtime(path)
            and os.path.getmtime(obj) > _newest_header()):
        return obj, ""
    cmd = [NVCC, *ARCH, *FLAGS, *EXTRA, "-x", "cu", "-c", path, "-o", obj]
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n{res.stdout}\n{res.stderr}")
    with open(obj + ".ptxas.txt", "w") as f:       # registers / spills / smem per kernel (-Xptxas -v)
        f.write(res.stderr)
    return obj, res.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJDIR, exist_ok=True)
    with cf.ThreadPoolExecutor(max_workers=min(8, len(SOURCES))) as ex:
        results = list(ex.map(lambda s: _compile(s, force, verbose), SOURCES))
    objs = [o for o, _ in results]
    if force or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        cmd = [NVCC, *ARCH, "-shared", "-o", LIB, *objs, "-lgomp"]
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="--verbose" in sys.argv or "-v" in sys.argv)
    print(LIB)
