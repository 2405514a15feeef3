"""Writes the stored oracle results tests/golden/cg_config<i>_<prec>.json for the large BASELINE
configs, where the fp64 CPU oracle takes minutes to an hour (32^4, 48^3x96).

It calls ONLY oracle/ (and the seeded input generators, which hold none of the method's arithmetic);
nothing here comes from the CUDA path.  Re-run with
    python tests/golden/make_golden.py 3:32 3:64 4:32
Each file stores: iteration count, recursed and true relative residual, the rr = <r,r> history, and
psi at a seeded sample of sites (so that a GPU solution can be compared element by element there).

The same for the solvers of the SURVEY.md 8(f3)/(f4) rows at full size (`rows:3:32 rows:3:64 rows:4:32` ->
tests/golden/rows_config<i>_fp<prec>.json): the oracle's BiCGSTAB on D (reading B1), its even-odd preconditioned
CG (E1) and its even-odd preconditioned BiCGSTAB (EB1), one record per solver in the same format.

prec = 32: inputs are the fp32-rounded fields promoted to fp64 (both sides then see the identical
operator and source); tolerance = the config's (1e-6).  prec = 64: unrounded
fp64 inputs, tolerance 1e-10 (BASELINE.json configs[3] "fp64 variant").
"""
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import wilson_oracle  # noqa: E402
from paper_2111_14958_b200 import inputs  # noqa: E402

N_SAMPLES = 96


def sample_sites(cfg_index, volume):
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([inputs.BASE_SEED, cfg_index, 77])))
    s = rng.choice(volume, size=N_SAMPLES - 2, replace=False)
    return np.sort(np.concatenate([[0, volume - 1], s])).astype(np.int64)


def tolerance(cfg, prec):
    return 1e-10 if prec == 64 else cfg.r_min


def make(cfg_index, prec):
    cfg = inputs.CONFIGS[cfg_index]
    t0 = time.time()
    dtype = np.complex64 if prec == 32 else np.complex128
    U, eta = inputs.config_inputs(cfg, dtype=dtype)
    U = U.astype(np.complex128)
    eta = eta.astype(np.complex128)
    t_gen = time.time() - t0
    r_min = tolerance(cfg, prec)
    psi, info = wilson_oracle.cg_solve(cfg.dims, U, eta, cfg.kappa, r_min, cfg.max_iter, cfg.bc_t, history=True)
    true_res = wilson_oracle.true_residual(cfg.dims, U, eta, psi, cfg.kappa, cfg.bc_t)
    sites = sample_sites(cfg_index, cfg.volume)
    ps = psi[sites].reshape(len(sites), 12)
    out = {
        "written_by": "tests/golden/make_golden.py (fp64 CPU oracle only)",
        "config": cfg_index, "name": cfg.name, "dims": list(cfg.dims), "kappa": cfg.kappa, "links": cfg.links,
        "bc_t": cfg.bc_t, "input_precision": prec, "r_min": r_min, "max_iter": cfg.max_iter,
        "iterations": info["iterations"], "converged": info["converged"],
        "rel_residual": info["rel_residual"], "true_residual": true_res, "eta_norm2": info["eta_norm2"],
        "oracle_seconds": info["seconds"], "oracle_threads": wilson_oracle.num_threads(), "gen_seconds": t_gen,
        "psi_norm2": wilson_oracle.norm2(psi),
        "rr_history": [float(v) for v in info["rr_history"]],
        "sample_sites": [int(s) for s in sites],
        "psi_samples_re": [[float(v) for v in row.real] for row in ps],
        "psi_samples_im": [[float(v) for v in row.imag] for row in ps],
    }
    path = os.path.join(HERE, f"cg_config{cfg_index}_fp{prec}.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=0)
    print(f"{path}: {info['iterations']} iterations, true residual {true_res:.3e}, "
          f"oracle {info['seconds']:.1f} s on {out['oracle_threads']} threads", flush=True)


ROW_SOLVERS = (("bicgstab", "bicgstab_solve"), ("cg_eo", "cg_solve_eo"), ("bicgstab_eo", "bicgstab_solve_eo"))


def make_rows(cfg_index, prec):
    """The oracle's solvers of the 8(f) rows on the same inputs, tolerance and iteration cap as `make`."""
    cfg = inputs.CONFIGS[cfg_index]
    dtype = np.complex64 if prec == 32 else np.complex128
    U, eta = inputs.config_inputs(cfg, dtype=dtype)
    U = U.astype(np.complex128)
    eta = eta.astype(np.complex128)
    r_min = tolerance(cfg, prec)
    sites = sample_sites(cfg_index, cfg.volume)
    out = {
        "written_by": "tests/golden/make_golden.py (fp64 CPU oracle only)",
        "config": cfg_index, "name": cfg.name, "dims": list(cfg.dims), "kappa": cfg.kappa, "links": cfg.links,
        "bc_t": cfg.bc_t, "input_precision": prec, "r_min": r_min, "max_iter": cfg.max_iter,
        "oracle_threads": wilson_oracle.num_threads(), "sample_sites": [int(s) for s in sites], "solvers": {},
    }
    path = os.path.join(HERE, f"rows_config{cfg_index}_fp{prec}.json")
    for name, fn in ROW_SOLVERS:
        psi, info = getattr(wilson_oracle, fn)(cfg.dims, U, eta, cfg.kappa, r_min, cfg.max_iter, cfg.bc_t, history=True)
        true_res = wilson_oracle.true_residual(cfg.dims, U, eta, psi, cfg.kappa, cfg.bc_t)
        ps = psi[sites].reshape(len(sites), 12)
        out["solvers"][name] = {
            "oracle_function": fn, "iterations": info["iterations"], "converged": info["converged"],
            "status": info["status"], "rel_residual": info["rel_residual"], "true_residual": true_res,
            "eta_norm2": info["eta_norm2"], "oracle_seconds": info["seconds"], "psi_norm2": wilson_oracle.norm2(psi),
            "rr_history": [float(v) for v in info["rr_history"]],
            "psi_samples_re": [[float(v) for v in row.real] for row in ps],
            "psi_samples_im": [[float(v) for v in row.imag] for row in ps],
        }
        print(f"{path}: {name}: {info['iterations']} iterations, true residual {true_res:.3e}, "
              f"oracle {info['seconds']:.1f} s on {out['oracle_threads']} threads", flush=True)
        del psi
        with open(path, "w") as f:      # rewritten after every solver: an interrupted run keeps what it finished
            json.dump(out, f, indent=0)


if __name__ == "__main__":
    for arg in sys.argv[1:] or ["3:32", "3:64", "4:32", "rows:3:32", "rows:3:64", "rows:4:32"]:
        if arg.startswith("rows:"):
            _, i, p = arg.split(":")
            make_rows(int(i), int(p))
        else:
            i, p = arg.split(":")
            make(int(i), int(p))
