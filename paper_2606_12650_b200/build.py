"""Build libnk.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_12650_b200.build [--force] [--verbose] | --census

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

SOURCES = ["nk_api.cu", "nk_setup.cu", "nk_plan.cu", "nk_ax_tma.cu", "nk_gs.cu", "nk_vec.cu", "nk_geom.cu", "nk_dist.cu", "nk_probe.cu", "nk_static.cu", "nk_basis.cpp"]
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


def census() -> str:
    """SASS / ptxas census of every kernel in libnk.so as a markdown table: registers and spill bytes (ptxas -v, kept
    beside the objects), and from `cuobjdump -sass` the counts of UBLKCP (bulk-copy / TMA engine), UBLKPF (bulk prefetch into L2), SYNCS (mbarrier),
    DFMA, DFMA with a uniform-register operand (D through the uniform datapath), LDL/STL (local memory), ACQBULK
    (griddepcontrol.wait), LDGSTS, and tensor-core MMA opcodes (none expected: fp64, HBM-bound)."""
    import re
    build()
    cuobjdump = os.path.join(os.path.dirname(NVCC), "cuobjdump")
    rows = []
    for src in SOURCES:
        if not src.endswith(".cu"):
            continue
        obj = os.path.join(OBJDIR, os.path.splitext(src)[0] + ".o")
        regs = {}
        try:
            txt = open(obj + ".ptxas.txt").read()
        except OSError:
            txt = ""
        for m in re.finditer(r"Compiling entry function '(\S+)'.*?\n.*?\n\s*(\d+) bytes stack frame, (\d+) bytes spill stores, "
                             r"(\d+) bytes spill loads\n.*?Used (\d+) registers", txt):
            regs[m.group(1)] = (int(m.group(5)), int(m.group(3)), int(m.group(4)))
        sass = subprocess.run([cuobjdump, "-sass", obj], capture_output=True, text=True).stdout
        name, counts = None, None

        def flush():
            if name is None:
                return
            dem = subprocess.run(["c++filt", name], capture_output=True, text=True).stdout.strip() or name
            dem = re.sub(r"\(anonymous namespace\)::", "", dem)
            dem = re.sub(r"\(.*", "", dem)[:60]
            r = regs.get(name, ("?", "?", "?"))
            rows.append((src, dem, r[0], f"{r[1]}/{r[2]}", counts["UBLKCP"], counts["UBLKPF"], counts["SYNCS"], counts["DFMA"], counts["DFMA_UR"],
                         counts["LDL"] + counts["STL"], counts["ACQBULK"], counts["MMA"]))
        for line in sass.splitlines():
            m = re.search(r"Function : (\S+)", line)
            if m:
                flush()
                name = m.group(1)
                counts = dict(UBLKCP=0, UBLKPF=0, SYNCS=0, DFMA=0, DFMA_UR=0, LDL=0, STL=0, ACQBULK=0, MMA=0)
                continue
            if counts is None or "/*" not in line:
                continue
            ins = line.split("*/", 1)[-1]
            for key in ("UBLKCP", "UBLKPF", "SYNCS", "ACQBULK"):
                if re.search(r"\b" + key, ins):
                    counts[key] += 1
            if re.search(r"\bDFMA\b", ins):
                counts["DFMA"] += 1
                if re.search(r"\bUR\d+", ins):
                    counts["DFMA_UR"] += 1
            if re.search(r"\bLDL\b|\bLDL\.", ins):
                counts["LDL"] += 1
            if re.search(r"\bSTL\b|\bSTL\.", ins):
                counts["STL"] += 1
            if re.search(r"\b(UTC\w*MMA|HMMA|DMMA|IMMA)\b", ins):
                counts["MMA"] += 1
        flush()
    out = ["| file | kernel | registers | spill B (st/ld) | UBLKCP | UBLKPF | SYNCS | DFMA | DFMA with UR operand | LDL+STL | ACQBULK | tensor MMA |",
           "|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for r in rows:
        out.append("| " + " | ".join(str(x) for x in r) + " |")
    return "\n".join(out)


if __name__ == "__main__":
    if "--census" in sys.argv:
        print(census())
    else:
        build(force="--force" in sys.argv, verbose="--verbose" in sys.argv or "-v" in sys.argv)
        print(LIB)
