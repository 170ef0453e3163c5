"""Build the CPU oracle shared library (test infrastructure): g++ -O2 -ffp-contract=off -fopenmp.

Run as `python oracle/build.py`; also called by `__graft_entry__.build()` and, lazily, by
`oracle/__init__.py` when the library is missing or older than its source."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "mrd_oracle.cpp")]
HDR = [os.path.join(HERE, "mrd_oracle.h")]
LIB = os.path.join(HERE, "libmrd_oracle.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SRC + HDR)


def build(force: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", tmp] + SRC
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
