"""Build step of the C-ABI library: nvcc, sm_100a only, in-tree (paper_2111_14958_b200/libwilson_cg.so).

`python -m paper_2111_14958_b200.build [--force] [-v]` or `__graft_entry__.build()`.  nvcc cross-compiles
without a GPU.  The translation units compile in parallel; objects and the .so are git-ignored and travel
to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libwilson_cg.so")
UNITS = ["wilson_cg.cu", "wilson_dslash_f32.cu", "wilson_dslash_f64.cu", "wilson_bicg_f32.cu", "wilson_bicg_f64.cu",
         "wilson_coo.cu", "wilson_eo.cu", "wilson_mrhs.cu", "wilson_mrhs_f32.cu", "wilson_mrhs_f64.cu", "wilson_dslash_eo_f32.cu", "wilson_dslash_eo_f64.cu", "wilson_dslash12_f32.cu", "wilson_dslash12_f64.cu",
         "wilson_bicg_eo_f32.cu", "wilson_bicg_eo_f64.cu", "wilson_split_f32.cu", "wilson_split_f64.cu",
         "wilson_dslash12_eo_f32.cu", "wilson_dslash12_eo_f64.cu",
         "wilson_eo_onelaunch_f32.cu", "wilson_eo_onelaunch_f64.cu",
         "wilson_dslash_y_f32.cu", "wilson_dslash_y_f64.cu"]
HEADERS = [os.path.join(CSRC, "wilson_kernels.cuh"), os.path.join(CSRC, "wilson_launch.cuh"),
           os.path.join(CSRC, "wilson_ctx.cuh"), os.path.join(CSRC, "wilson_mrhs.cuh"), os.path.join(CSRC, "wilson_split.cuh"), os.path.join(CSRC, "wilson_eo_onelaunch.cuh"),
           os.path.join(ROOT, "include", "wilson_cg.h")]

ARCH_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ["-std=c++17", "-O3", "-lineinfo"] + ARCH_FLAGS + ["-Xcompiler", "-fPIC"]


def nvcc_path() -> str:
    cand = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    return cand if os.path.exists(cand) else "nvcc"


def _stale(target, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libwilson_cg.so if missing or older than its sources.  Returns its path."""
    os.makedirs(OBJDIR, exist_ok=True)
    objs, jobs = [], []
    for unit in UNITS:
        src = os.path.join(CSRC, unit)
        obj = os.path.join(OBJDIR, unit.replace(".cu", ".o"))
        objs.append(obj)
        if force or _stale(obj, [src] + HEADERS):
            cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
            jobs.append(cmd)
    if jobs:
        with ThreadPoolExecutor(len(jobs)) as pool:
            for rc, cmd in zip(pool.map(lambda c: subprocess.run(c, cwd=CSRC).returncode, jobs), jobs):
                if rc != 0:
                    raise RuntimeError("nvcc failed: " + " ".join(cmd))
    if jobs or force or _stale(LIB, objs):
        tmp = LIB + f".{os.getpid()}.tmp"
        subprocess.check_call([nvcc_path()] + ARCH_FLAGS + ["--shared", "-o", tmp] + objs)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
