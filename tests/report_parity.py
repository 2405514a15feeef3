"""Prints the parity table of BASELINE.md section 3 (GPU vs fp64 CPU oracle on the five BASELINE configs).
Test-side script (it imports the oracle); run on a GPU box:  python tests/report_parity.py [max_config]
For configs 3 and 4 the oracle's CG result comes from tests/golden/*.json (written by make_golden.py); the
per-site operator errors and the true residual of the GPU solution are evaluated live by the oracle."""
import json
import os
import sys

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)

from oracle import wilson_oracle  # noqa: E402
from paper_2111_14958_b200 import inputs, wilson  # noqa: E402
import lattice_math as lm  # noqa: E402


def main(max_cfg=4):
    print("| config | precision | wd_apply D err (site max) | D-dagger err | iterations GPU / oracle | "
          "true residual GPU / oracle | recursed residual GPU |")
    print("|---|---|---|---|---|---|---|")
    for ci, prec in ((0, 32), (1, 32), (2, 32), (3, 32), (3, 64), (4, 32)):
        if ci > max_cfg:
            continue
        cfg = inputs.CONFIGS[ci]
        r_min = cfg.r_min if prec == 32 else 1e-10
        cdt = np.complex64 if prec == 32 else np.complex128
        U, eta = inputs.config_inputs(cfg, dtype=cdt)
        U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
        with wilson.WilsonContext(cfg.dims, prec, cfg.bc_t) as ctx:
            Un = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
            en = ctx.wd_pack_spinor(torch.from_numpy(eta).cuda())
            errs = []
            rng = np.random.Generator(np.random.PCG64(1))
            sites = np.unique(np.concatenate([[0, cfg.volume - 1], rng.choice(cfg.volume, min(cfg.volume, 20000), replace=False)]))
            for dag in (False, True):
                got = ctx.wd_unpack_spinor(ctx.wd_apply(Un, en, cfg.kappa, dag)).cpu().numpy()[sites]
                want = wilson_oracle.wd_apply_sites(cfg.dims, U64, eta64, cfg.kappa, sites, dag, cfg.bc_t)
                errs.append(lm.per_site_rel_err(got, want)[0])
            psi_n, info = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter)
            psi = ctx.wd_unpack_spinor(psi_n).cpu().numpy().astype(np.complex128)
        res = wilson_oracle.true_residual(cfg.dims, U64, eta64, psi, cfg.kappa, cfg.bc_t)
        gold = os.path.join(HERE, "golden", f"cg_config{ci}_fp{prec}.json")
        if os.path.exists(gold):
            g = json.load(open(gold))
            it_o, res_o = g["iterations"], g["true_residual"]
        else:
            psi_o, info_o = wilson_oracle.cg_solve(cfg.dims, U64, eta64, cfg.kappa, r_min, cfg.max_iter, cfg.bc_t)
            it_o = info_o["iterations"]
            res_o = wilson_oracle.true_residual(cfg.dims, U64, eta64, psi_o, cfg.kappa, cfg.bc_t)
        print(f"| {ci}: {cfg.name} | fp{prec} | {errs[0]:.2e} | {errs[1]:.2e} | {info['iterations']} / {it_o} | "
              f"{res:.3e} / {res_o:.3e} | {info['rel_residual']:.3e} |", flush=True)


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 4)
