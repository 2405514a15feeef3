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


def rows(max_cfg=4):
    """The SURVEY.md 8(f) rows: BiCGSTAB, even-odd CG, 12-real CG (iterations and true residual, GPU / oracle) and the
    COO route.  The oracle solves run live for configs 0-2; at configs 3 and 4 only the true residual of the GPU
    solution is evaluated (one oracle D application)."""
    print("\n| config | solver | iterations GPU / oracle | true residual GPU / oracle |")
    print("|---|---|---|---|")
    for ci in range(0, max_cfg + 1):
        cfg = inputs.CONFIGS[ci]
        U, eta = inputs.config_inputs(cfg, dtype=np.complex64)
        U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
        live = ci <= 2
        with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
            Ud, ed = torch.from_numpy(U).cuda(), torch.from_numpy(eta).cuda()
            Un, en = ctx.wd_pack_gauge(Ud), ctx.wd_pack_spinor(ed)
            out = {}
            pn, ib = ctx.bicgstab_solve(Un, en, cfg.kappa, cfg.r_min, cfg.max_iter)
            out["BiCGSTAB on D"] = (ctx.wd_unpack_spinor(pn).cpu().numpy(), ib, wilson_oracle.bicgstab_solve)
            Ue, ee = ctx.wd_eo_pack_gauge(Ud), ctx.wd_eo_pack_spinor(ed)
            pe, ie = ctx.cg_solve_eo(Ue, ee, cfg.kappa, cfg.r_min, cfg.max_iter)
            out["even-odd CG"] = (ctx.wd_eo_unpack_spinor(pe).cpu().numpy(), ie, wilson_oracle.cg_solve_eo)
            pe, ieb = ctx.bicgstab_solve_eo(Ue, ee, cfg.kappa, cfg.r_min, cfg.max_iter)
            out["even-odd BiCGSTAB"] = (ctx.wd_eo_unpack_spinor(pe).cpu().numpy(), ieb, wilson_oracle.bicgstab_solve_eo)
            del Ue, ee, pe
            ctx.wd_set_gauge_recon(12)
            p12, i12 = ctx.cg_solve(ctx.wd_pack_gauge(Ud), en, cfg.kappa, cfg.r_min, cfg.max_iter)
            out["CG, 12-real links"] = (ctx.wd_unpack_spinor(p12).cpu().numpy(), i12, wilson_oracle.cg_solve)
        for name, (psi, info, ofun) in out.items():
            res = wilson_oracle.true_residual(cfg.dims, U64, eta64, psi.astype(np.complex128), cfg.kappa, cfg.bc_t)
            if live:
                po, io = ofun(cfg.dims, U64, eta64, cfg.kappa, cfg.r_min, cfg.max_iter, cfg.bc_t)
                ro = wilson_oracle.true_residual(cfg.dims, U64, eta64, po, cfg.kappa, cfg.bc_t)
                print(f"| {ci}: {cfg.name} | {name} | {info['iterations']} / {io['iterations']} | {res:.3e} / {ro:.3e} |", flush=True)
            else:
                print(f"| {ci}: {cfg.name} | {name} | {info['iterations']} / (not run) | {res:.3e} / — |", flush=True)
    # COO at 14^4
    cfg = inputs.CONFIGS[2]
    U, eta = inputs.config_inputs(cfg, dtype=np.complex64)
    with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
        Un = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
        val, row, col = ctx.wd_coo_assemble(Un, cfg.kappa, False)
        got = ctx.wd_coo_spmv(val, row, col, torch.from_numpy(eta).cuda()).cpu().numpy()
    want = wilson_oracle.wd_apply(cfg.dims, U.astype(np.complex128), eta.astype(np.complex128), cfg.kappa, False, cfg.bc_t)
    print(f"\nCOO SpMV at 14^4 (N_NZ = {val.numel()}): per-site relative error against the oracle's D "
          f"{lm.per_site_rel_err(got, want)[0]:.2e}", flush=True)


if __name__ == "__main__":
    mc = int(sys.argv[1]) if len(sys.argv) > 1 else 4
    main(mc)
    rows(mc)
