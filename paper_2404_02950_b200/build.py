"""Build libsledge.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2404_02950_b200.build [--force]

FMA contraction is disabled (--fmad=false) so that every product and sum is individually rounded, which
is what the string-tag rule requires (R8) and what keeps the field arithmetic comparable with
the oracle rounding for rounding; the path is HBM-bound, the extra instructions are free.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsledge.so")
SOURCES = ["sledge.cu"]
DEPS = ["sledge.cu", "layout.h", "k_rk_pipe.cuh", "k_rk_plane.cuh", "k_rk_tma.cuh", "k_gw.cuh", "k_ghost.cuh", "k_tag.cuh",
        "k_avgdown.cuh",
        os.path.join("..", "..", "include", "sledge.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--fmad=false",
              "-shared", "-Xcompiler", "-fPIC"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
        subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
