"""Build oracle/libsie_dfmp2_oracle.so (plain C, gcc). Test infrastructure only.

Usage: python oracle/build.py   (also called by __graft_entry__.build()).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dfmp2_oracle.c")
LIB = os.path.join(HERE, "libsie_dfmp2_oracle.so")
# x86-64-v3 (AVX2+FMA) rather than -march=native: the .so built in one container must also run on the GPU box.
CFLAGS = ["-O3", "-march=x86-64-v3", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", *CFLAGS, "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
