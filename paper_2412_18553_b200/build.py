"""Build paper_2412_18553_b200/libsie_dfmp2.so in-tree with nvcc for sm_100a.

Usage: python -m paper_2412_18553_b200.build [--force]   (also called by __graft_entry__.build()).
nvcc cross-compiles without a GPU; the static CUDA runtime is linked, libcuda is NOT (the one driver entry
point needed, cuTensorMapEncodeTiled, is fetched at run time), so the library loads on a CPU-only host.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsie_dfmp2.so")
SOURCES = ["api.cu", "transform.cu", "pair.cu", "general.cu", "canonical.cu", "noalloc.cu", "ref_kernels.cu", "probes.cu"]
HEADERS = ["sie_common.cuh", "mma_pipeline.cuh", "sie_internal.h", os.path.join("..", "..", "include", "sie_dfmp2.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "static",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("SIE_NVCC_EXTRA", "").split()  # e.g. -DSIE_EXP_...=1 for kernel experiments
    cmd = [nvcc, *NVCC_FLAGS, *extra, *( ["-Xptxas", "-v"] if verbose else []), "-o", LIB, *[os.path.join(CSRC, f) for f in SOURCES]]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
