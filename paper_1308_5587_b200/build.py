"""Build libhb.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1308_5587_b200.build [--force]

No torch involved: the library links only against the CUDA runtime.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhb.so")
SOURCES = ["hb_api.cu", "cells.cu", "nlist.cu", "force.cu", "nve.cu", "sort.cu", "peaks.cu", "dp.cu", "thermo_static.cu"]
HEADERS = [os.path.join(CSRC, n) for n in ("hb_internal.cuh", "tile.cuh", "cells_dev.cuh", "integrate_dev.cuh")] + \
          [os.path.join(os.path.dirname(HERE), "include", "hb.h")]

# IEEE arithmetic throughout: no --use_fast_math.  The cell index and the grid
# coordinate use explicit __fsub_rn/__fmul_rn so that contraction cannot touch them.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--threads", "0"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    cmd = [nvcc(), *NVCC_FLAGS, *os.environ.get("HB_NVCC_EXTRA", "").split(), "-shared", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES] + ["-ldl"]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(LIB)
