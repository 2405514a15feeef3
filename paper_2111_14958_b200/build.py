"""Build step of the C-ABI library: nvcc, sm_100a only, in-tree (paper_2111_14958_b200/libwilson_cg.so).

`python -m paper_2111_14958_b200.build [--force]` or `__graft_entry__.build()`.  nvcc cross-compiles
without a GPU.  The .so is git-ignored and travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libwilson_cg.so")
SOURCES = [os.path.join(CSRC, "wilson_cg.cu")]
DEPENDS = SOURCES + [os.path.join(CSRC, "wilson_kernels.cuh"), os.path.join(ROOT, "include", "wilson_cg.h")]

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "--shared", "-Xcompiler", "-fPIC",
    "--threads", "0",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in DEPENDS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libwilson_cg.so if missing or older than its sources.  Returns its path."""
    if force or is_stale():
        tmp = LIB + f".{os.getpid()}.tmp"
        cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        subprocess.check_call(cmd, cwd=CSRC)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
