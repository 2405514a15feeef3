"""Build step of the C-ABI library: nvcc, sm_100a only, in-tree (paper_2111_14958_b200/libwilson_cg.so).

`python -m paper_2111_14958_b200.build [--force] [-v]` or `__graft_entry__.build()`.  nvcc cross-compiles
without a GPU.  The translation units compile in parallel; objects and the .so are git-ignored and travel
to the GPU box with the gpurun snapshot.

An object is reused only if `build/manifest.json` records, for it, the SHA-256 of exactly the sources it
was compiled from (its .cu, every header, the nvcc command line and the nvcc version); anything else is
recompiled.  Every call prints one line saying how many units were compiled and how many reused, and
`last_report()` returns the same as a dict, so that a prebuilt binary riding along with a snapshot is visible
as such (and provably the product of the sources beside it).
"""
from __future__ import annotations

import hashlib
import json
import os
import subprocess
import sys
import time
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libwilson_cg.so")
MANIFEST = os.path.join(OBJDIR, "manifest.json")
UNITS = ["wilson_cg.cu", "wilson_dslash_f32.cu", "wilson_dslash_f64.cu", "wilson_bicg_f32.cu", "wilson_bicg_f64.cu",
         "wilson_coo.cu", "wilson_eo.cu", "wilson_mrhs.cu", "wilson_mrhs_f32.cu", "wilson_mrhs_f64.cu",
         "wilson_dslash_eo_f32.cu", "wilson_dslash_eo_f64.cu", "wilson_dslash12_f32.cu", "wilson_dslash12_f64.cu",
         "wilson_bicg_eo_f32.cu", "wilson_bicg_eo_f64.cu", "wilson_split_f32.cu", "wilson_split_f64.cu",
         "wilson_dslash12_eo_f32.cu", "wilson_dslash12_eo_f64.cu",
         "wilson_eo_onelaunch_f32.cu", "wilson_eo_onelaunch_f64.cu", "wilson_tma_f32.cu", "wilson_tma_f64.cu",
         "wilson_resident_f32.cu", "wilson_resident_f64.cu", "wilson_ures_f32.cu", "wilson_ures_f64.cu",
         "wilson_noalloc.cu"]

ARCH_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a"]
# --compress-mode=size: the SASS of the ~500 template instantiations compresses about tenfold (the library went from
# 76 MB to under 10 MB); the driver inflates it when the module is loaded
NVCC_FLAGS = ["-std=c++17", "-O3", "-lineinfo", "--compress-mode=size"] + ARCH_FLAGS + ["-Xcompiler", "-fPIC"]

_last_report: dict = {}


def nvcc_path() -> str:
    cand = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    return cand if os.path.exists(cand) else "nvcc"


def _headers():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")) + \
        [os.path.join(ROOT, "include", "wilson_cg.h")]


def _sha(paths, extra=""):
    h = hashlib.sha256(extra.encode())
    for p in paths:
        with open(p, "rb") as f:
            h.update(hashlib.sha256(f.read()).digest())
    return h.hexdigest()


def _nvcc_version() -> str:
    try:
        return subprocess.run([nvcc_path(), "--version"], capture_output=True, text=True).stdout.strip().splitlines()[-1]
    except OSError:
        return "unknown"


def last_report() -> dict:
    """What the last build() call of this process did: {'compiled': [...], 'reused': [...], 'linked': bool, ...}"""
    return dict(_last_report)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libwilson_cg.so unless every object and the library are the product of the present sources."""
    t0 = time.time()
    os.makedirs(OBJDIR, exist_ok=True)
    try:
        with open(MANIFEST) as f:
            manifest = json.load(f)
    except (OSError, ValueError):
        manifest = {}
    headers = _headers()
    flags = " ".join(NVCC_FLAGS) + " | " + _nvcc_version()
    hdr_sha = _sha(headers, flags)
    objs, jobs, want = [], [], {}
    for unit in UNITS:
        src = os.path.join(CSRC, unit)
        obj = os.path.join(OBJDIR, unit.replace(".cu", ".o"))
        objs.append(obj)
        want[unit] = _sha([src], hdr_sha)
        if force or not os.path.exists(obj) or manifest.get("units", {}).get(unit) != want[unit]:
            jobs.append((unit, [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]))
    if jobs:
        workers = max(1, min(len(jobs), os.cpu_count() or 4))
        with ThreadPoolExecutor(workers) as pool:
            for rc, (unit, cmd) in zip(pool.map(lambda j: subprocess.run(j[1], cwd=CSRC).returncode, jobs), jobs):
                if rc != 0:
                    raise RuntimeError("nvcc failed: " + " ".join(cmd))
    lib_key = _sha([], "".join(want[u] for u in UNITS))
    link = bool(jobs) or force or not os.path.exists(LIB) or manifest.get("lib") != lib_key
    if link:
        tmp = LIB + f".{os.getpid()}.tmp"
        subprocess.check_call([nvcc_path()] + ARCH_FLAGS + ["--shared", "-o", tmp] + objs)
        os.replace(tmp, LIB)
    with open(MANIFEST, "w") as f:
        json.dump({"units": want, "lib": lib_key, "flags": flags}, f, indent=0)
    compiled = [u for u, _ in jobs]
    _last_report.clear()
    _last_report.update({"compiled": compiled, "reused": [u for u in UNITS if u not in compiled], "linked": link,
                         "seconds": round(time.time() - t0, 1), "lib_bytes": os.path.getsize(LIB), "flags": flags})
    print(f"[build] libwilson_cg.so: compiled {len(compiled)} of {len(UNITS)} translation units, reused "
          f"{len(UNITS) - len(compiled)} (source hashes match build/manifest.json), "
          f"{'linked' if link else 'library up to date'}, {_last_report['lib_bytes'] / 1e6:.1f} MB, "
          f"{_last_report['seconds']} s", file=sys.stderr, flush=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
