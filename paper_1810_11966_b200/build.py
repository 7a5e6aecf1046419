"""Builds libcbmtrigger.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1810_11966_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the tree.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libcbmtrigger.so")
SOURCES = [os.path.join(CSRC, "cbm_trigger.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "ptx.cuh"), os.path.join(CSRC, "classify.cuh"), os.path.join(CSRC, "tile.cuh"), os.path.join(CSRC, "team.cuh"), os.path.join(CSRC, "select.cuh"), os.path.join(CSRC, "wire.cuh"), os.path.join(CSRC, "msd.cuh"), os.path.join(CSRC, "filter.cuh"), os.path.join(CSRC, "ubench.cuh"), os.path.join(CSRC, "chain.cuh"), os.path.join(CSRC, "timeslice.cuh"), os.path.join(CSRC, "params.h"),
                  os.path.join(INCLUDE, "cbm_trigger.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build_library(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
        subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
