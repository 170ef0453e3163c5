"""Build the CUDA library `libmrd.so` in-tree for sm_100a (nvcc cross-compiles without a GPU).

Run as `python -m paper_1705_02028_b200.build [--force] [--verbose]`; also called by
`__graft_entry__.build()` and lazily by the binding when the library is missing or stale."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INC = os.path.join(os.path.dirname(HERE), "include")
SRC = [os.path.join(CSRC, "mrd_api.cu"), os.path.join(CSRC, "mrd_meshgen.cu"), os.path.join(CSRC, "mrd_layout.cpp"),
       os.path.join(CSRC, "mrd_partition.cpp")]
DEPS = SRC + [os.path.join(CSRC, f) for f in ("mrd_kernels.cuh", "mrd_tile.cuh", "mrd_math.cuh", "mrd_layout.h", "mrd_predicates.cuh")] + [
    os.path.join(INC, "mrd.h")]
LIB = os.path.join(HERE, "libmrd.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-fopenmp,-O2", "-shared", "-lgomp"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SRC
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
