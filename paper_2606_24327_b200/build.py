"""Build libtrimeg_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

  python -m paper_2606_24327_b200.build [--force] [-v] [--defs "-DNAME=VALUE ..."]

`--defs` is for tuning builds only (TRIMEG_NCOMP, TRIMEG_NSLOTS, TRIMEG_WAITSTATS, ...; see csrc/trimeg_tile.cuh and
csrc/trimeg_ws.cuh).  Whatever was passed is compiled into the library and reported by trimeg_build_info(), so that a
benchmark line can never come from a non-default build unnoticed.  The environment is not consulted.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtrimeg_b200.so")
SOURCES = ["trimeg.cu"]
DEPS = ["trimeg.cu", "trimeg_kernels.cuh", "trimeg_ws.cuh", "trimeg_gather.cuh", "trimeg_math.cuh", "trimeg_host_setup.hpp", "trimeg_tile.cuh",
        "../../include/trimeg.h"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC", "-shared"]


def nvcc_path() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for d in DEPS:
        f = os.path.normpath(os.path.join(CSRC, d))
        if os.path.exists(f) and os.path.getmtime(f) > t:
            return True
    return False


def build(force: bool = False, verbose: bool = False, extra=(), defs: str = "") -> str:
    if not force and not defs and not stale():
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    info = '-DTRIMEG_BUILD_DEFS="' + defs.replace('"', "'") + '"'
    cmd = [nvcc_path(), *NVCC_FLAGS, *defs.split(), info, *extra, "-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        print(" ".join(cmd), flush=True)
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    argv = sys.argv[1:]
    defs = argv[argv.index("--defs") + 1] if "--defs" in argv else ""
    print(build(force="--force" in argv, verbose=True, extra=["-Xptxas", "-v"] if "-v" in argv else [], defs=defs))
