"""Measurement tables of BASELINE.md (not the bench line: that is bench.py at the repo root).

    python -m paper_2111_14958_b200.measure --report            one JSON line per BASELINE config: wd_apply D / D-dagger
                                                                over 100 applications, the CG solve
    python -m paper_2111_14958_b200.measure --rows              one JSON line per SURVEY.md 8(f) row (12-real links, BiCGSTAB,
                                                                even-odd solvers at configs 3 and 4, the COO SpMV)
    python -m paper_2111_14958_b200.measure --sweep --config I  every compiled launch configuration (the paper's
                                                                workgroup-size tuning) on config I
    python -m paper_2111_14958_b200.measure --staging --config I [--precision 64] [--reps N]
                                                                the stencil with the shared-memory link pipeline
                                                                (wd_set_link_staging, csrc/wilson_tma.cuh): every compiled
                                                                row that covers config I beside the kernel that reads the
                                                                links through L1, a2 / a3 / a4 inside the CG loop and wd_apply

All of it runs through the C-ABI binding (wilson.py) on seeded synthetic lattices (inputs.py); nothing here touches the
CPU oracle.  Needs a CUDA device.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

from . import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FLOP_ITER = 2976        # per site per CG iteration (reading G14)
FLOP_APPLY = 1368       # per site per D / D-dagger application
BYTES_ITER = {32: 1536, 64: 3072}  # a2 + a3 + a4


def cg_flops(volume, iterations):
    return float(volume) * (FLOP_ITER * iterations + FLOP_APPLY)


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def time_wd_apply(ctx, Un, en, out, kappa, dagger, reps=100):
    """device time per application over `reps` back-to-back applications (enqueued from C by wd_apply_repeat, CUDA
    events on the ctx stream; median of three rounds)"""
    return sorted(ctx.wd_apply_repeat(Un, en, kappa, dagger, reps, out=out) for _ in range(3))[1]


def run_report(args):
    """every config, wd_apply D and D-dagger (100 applications each, BASELINE.json configs[2])
    and the whole CG solve."""
    import torch

    from . import build as wbuild
    from . import wilson

    wbuild.build()
    wilson.load_library()
    for ci, prec in ((0, 32), (1, 32), (2, 32), (3, 32), (3, 64), (4, 32)):
        cfg = inputs.CONFIGS[ci]
        r_min = cfg.r_min if prec == 32 else 1e-10
        U, eta = inputs.config_inputs(cfg, dtype=np.complex64 if prec == 32 else np.complex128)
        V = cfg.volume
        with wilson.WilsonContext(cfg.dims, prec, cfg.bc_t) as ctx:
            Un = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
            en = ctx.wd_pack_spinor(torch.from_numpy(eta).cuda())
            out = ctx.empty_spinor()
            d_ms = time_wd_apply(ctx, Un, en, out, cfg.kappa, False)
            dd_ms = time_wd_apply(ctx, Un, en, out, cfg.kappa, True)
            for _ in range(2):
                ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
            ctx.wd_set_profile(True)
            ms = []
            for _ in range(3):
                _, info = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
                ms.append(info["gpu_ms"])
            prof = ctx.wd_get_profile()
            t = float(np.median(ms))
            it = info["iterations"]
            bpi = BYTES_ITER[prec]
            iter_ms = (prof["a2_ms"] + prof["a3_ms"] + prof["a4_ms"]) / prof["iterations"] if prof["iterations"] else None
            print(json.dumps({
                "report": f"config{ci}", "name": cfg.name, "precision": prec, "volume": V,
                "wd_apply_D_us": d_ms * 1e3, "wd_apply_Ddag_us": dd_ms * 1e3, "applications": 100,
                "wd_apply_D_gflops": FLOP_APPLY * V / (d_ms * 1e-3) / 1e9,
                "wd_apply_Ddag_gflops": FLOP_APPLY * V / (dd_ms * 1e-3) / 1e9,
                "wd_apply_D_gflops_hopping_only_1320": 1320 * V / (d_ms * 1e-3) / 1e9,
                "wd_apply_Ddag_gflops_hopping_only_1320": 1320 * V / (dd_ms * 1e-3) / 1e9,
                "wd_apply_D_gbs": (480 if prec == 32 else 960) * V / (d_ms * 1e-3) / 1e9,
                "cg_iterations": it, "cg_rel_residual": info["rel_residual"], "cg_mode": info["cg_mode"],
                "cg_solve_ms": t, "cg_gflops": cg_flops(V, it) / (t * 1e-3) / 1e9,
                "cg_us_per_iteration": t / max(it, 1) * 1e3,
                "cg_iteration_gbs_live": bpi * V / (iter_ms * 1e-3) / 1e9 if iter_ms else None,
                "cg_iteration_gbs_whole_solve": bpi * V * it / (t * 1e-3) / 1e9,
                "tile": list(wilson.tile_shapes()[ctx.wd_get_tile()])}), flush=True)
    return 0


FLOP_BICG_ITER = 2 * 1368 + 960   # two D applications + 10 complex vector/dot operations
BYTES_BICG = {32: (576, 288, 480, 672, 384), 64: (1152, 576, 960, 1344, 768)}   # the five kernels of one iteration
FLOP_COO_NNZ = 8                   # one complex multiply-add per stored entry
NNZ_PER_SITE = 588


def run_rows(args):
    """The SURVEY.md 8(f) rows, one JSON line each: BiCGSTAB (f4) and 12-real links (f3) at configs 3 and 4, the paper's
    COO SpMV (f2) at 14^4 (config 2, the largest volume of the paper's range) beside the matrix-free stencil."""
    import torch

    from . import build as wbuild
    from . import wilson

    wbuild.build()
    wilson.load_library()
    peak, _ = measured_peak()
    prec = args.precision
    cdt = np.complex64 if prec == 32 else np.complex128
    rb = 4 if prec == 32 else 8
    for ci in [int(x) for x in args.rows_configs.split(",") if x]:
        cfg = inputs.CONFIGS[ci]
        r_min = cfg.r_min if prec == 32 else 1e-10
        U, eta = inputs.config_inputs(cfg, dtype=cdt)
        V = cfg.volume
        for recon in (18, 12):
            with wilson.WilsonContext(cfg.dims, prec, cfg.bc_t) as ctx:
                ctx.wd_set_gauge_recon(recon)
                Un = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
                en = ctx.wd_pack_spinor(torch.from_numpy(eta).cuda())
                out = ctx.empty_spinor()
                d_ms = time_wd_apply(ctx, Un, en, out, cfg.kappa, False)
                for _ in range(2):
                    ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
                ctx.wd_set_profile(True)
                ms = []
                for _ in range(3):
                    _, info = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
                    ms.append(info["gpu_ms"])
                p = ctx.wd_get_profile()
                ctx.wd_set_profile(False)
                n = max(p["iterations"], 1)
                gb = (72 if recon == 18 else 48) * rb          # gauge bytes per site
                sb = 24 * rb                                    # spinor bytes per site
                b2, b3, b4 = 2 * sb + gb, 3 * sb + gb, 5 * sb
                a2, a3, a4 = p["a2_ms"] / n, p["a3_ms"] / n, p["a4_ms"] / n
                t = float(np.median(ms))
                gbs = lambda b, msec: b * V / (msec * 1e-3) / 1e9 if msec > 0 else None
                print(json.dumps({
                    "row": "f3 link storage", "config": ci, "precision": prec, "reals_per_link": recon,
                    "bytes_per_site": {"wd_apply": b2, "a2": b2, "a3": b3, "a4": b4, "cg_iteration": b2 + b3 + b4},
                    "wd_apply_D_us": d_ms * 1e3, "wd_apply_D_gbs": b2 * V / (d_ms * 1e-3) / 1e9,
                    "cg_iterations": info["iterations"], "cg_solve_ms": t,
                    "cg_gflops": cg_flops(V, info["iterations"]) / (t * 1e-3) / 1e9,
                    "a2_us": a2 * 1e3, "a3_us": a3 * 1e3, "a4_us": a4 * 1e3,
                    # one-launch solves (small volumes) have no per-kernel times: the rates are then null
                    "a2_gbs": gbs(b2, a2), "a3_gbs": gbs(b3, a3),
                    "cg_iteration_gbs": gbs(b2 + b3 + b4, a2 + a3 + a4),
                    "cg_iteration_frac_of_measured": (gbs(b2 + b3 + b4, a2 + a3 + a4) or 0.0) / peak or None}), flush=True)
                if recon == 18:
                    for _ in range(2):
                        ctx.bicgstab_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
                    ctx.wd_set_profile(True)
                    ms = []
                    for _ in range(5):
                        _, ib = ctx.bicgstab_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
                        ms.append(ib["gpu_ms"])
                    pb = ctx.wd_get_profile_bicgstab()
                    ctx.wd_set_profile(False)
                    kus = [m / max(pb["iterations"], 1) * 1e3 for m in pb["ms"]]
                    bb = BYTES_BICG[prec]
                    tb = float(np.median(ms))
                    print(json.dumps({
                        "row": "f4 bicgstab", "config": ci, "precision": prec, "iterations": ib["iterations"],
                        "status": ib["status"], "rel_residual": ib["rel_residual"], "solve_ms": tb,
                        "gflops": FLOP_BICG_ITER * V * ib["iterations"] / (tb * 1e-3) / 1e9,
                        "kernel_us": dict(zip(("Dp_rv", "s", "Ds_ts", "xr", "p"), kus)),
                        "kernel_gbs": dict(zip(("Dp_rv", "s", "Ds_ts", "xr", "p"),
                                               [b * V / (u * 1e-6) / 1e9 if u > 0 else None for b, u in zip(bb, kus)])),
                        "iteration_gbs": sum(bb) * V / (sum(kus) * 1e-6) / 1e9 if sum(kus) > 0 else None,
                        "iteration_frac_of_measured": sum(bb) * V / (sum(kus) * 1e-6) / 1e9 / peak if sum(kus) > 0 else None,
                        "cg_solve_ms_same_problem": t, "speedup_vs_cg": t / tb}), flush=True)
                if recon == 18:
                    for nrhs in (2, 4):
                        em = torch.stack([en * (1.0 + 0.25 * j) for j in range(nrhs)]).contiguous()
                        om = ctx.empty_multi_spinor(nrhs)
                        for _ in range(3):
                            ctx.wd_apply_multi(Un, em, cfg.kappa, False, out=om)
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        torch.cuda.synchronize()
                        e0.record()
                        for _ in range(20):
                            ctx.wd_apply_multi(Un, em, cfg.kappa, False, out=om)
                        e1.record()
                        torch.cuda.synchronize()
                        ap_ms = e0.elapsed_time(e1) / 20
                        ctx.cg_solve_multi(Un, em, cfg.kappa, r_min, cfg.max_iter, out=om)
                        ctx.wd_set_profile(True)
                        _, infos = ctx.cg_solve_multi(Un, em, cfg.kappa, r_min, cfg.max_iter, out=om)
                        pm = ctx.wd_get_profile_bicgstab()
                        ctx.wd_set_profile(False)
                        km = [m / max(pm["iterations"], 1) * 1e3 / nrhs for m in pm["ms"][:3]]
                        bm = (2 * sb + gb / nrhs, 3 * sb + gb / nrhs, 5 * sb)     # per source: the links are shared
                        print(json.dumps({
                            "row": "f3 multi-rhs", "config": ci, "precision": prec, "nrhs": nrhs,
                            "iterations": [i["iterations"] for i in infos],
                            "wd_apply_us_per_source": ap_ms * 1e3 / nrhs, "wd_apply_us_single": d_ms * 1e3,
                            "solve_ms_per_source": infos[0]["gpu_ms"] / nrhs, "solve_ms_single": t,
                            "kernel_us_per_source": dict(zip(("a2", "a3", "a4"), km)),
                            "bytes_per_site_per_source": dict(zip(("a2", "a3", "a4"), bm)),
                            "iteration_gbs": sum(bm) * V / (sum(km) * 1e-6) / 1e9 if sum(km) > 0 else None,
                            "speedup_per_source_vs_single": t / (infos[0]["gpu_ms"] / nrhs)}), flush=True)
                        del em, om
                    Ue = ctx.wd_eo_pack_gauge(torch.from_numpy(U).cuda())
                    ee = ctx.wd_eo_pack_spinor(torch.from_numpy(eta).cuda())
                    pe = ctx.empty_eo_spinor()
                    for _ in range(2):
                        ctx.cg_solve_eo(Ue, ee, cfg.kappa, r_min, cfg.max_iter, out=pe)
                    ctx.wd_set_profile(True)
                    ms = []
                    for _ in range(5):
                        _, ie = ctx.cg_solve_eo(Ue, ee, cfg.kappa, r_min, cfg.max_iter, out=pe)
                        ms.append(ie["gpu_ms"])
                    pb = ctx.wd_get_profile_bicgstab()
                    ctx.wd_set_profile(False)
                    kus = [m / max(pb["iterations"], 1) * 1e3 for m in pb["ms"]]
                    # bytes per FULL-lattice site: each half-lattice pass reads the whole gauge field (forward links of
                    # its own parity, backward links of the other) and half-length spinors
                    hb = (sb // 2 + gb + sb // 2, sb // 2 + gb + sb, sb // 2 + gb + sb // 2, sb // 2 + gb + sb // 2 + sb,
                          5 * sb // 2)
                    te = float(np.median(ms))
                    names = ("Hdag_oe", "Mdag_qq", "H_oe", "M_rupd", "axpy")
                    print(json.dumps({
                        "row": "f3 even-odd cg", "config": ci, "precision": prec, "iterations": ie["iterations"],
                        "status": ie["status"], "rel_residual": ie["rel_residual"], "solve_ms": te,
                        "kernel_us": dict(zip(names, kus)), "bytes_per_full_site": dict(zip(names, hb)),
                        "kernel_gbs": dict(zip(names, [b * V / (u * 1e-6) / 1e9 if u > 0 else None for b, u in zip(hb, kus)])),
                        "iteration_gbs": sum(hb) * V / (sum(kus) * 1e-6) / 1e9 if sum(kus) > 0 else None,
                        "iteration_frac_of_measured": sum(hb) * V / (sum(kus) * 1e-6) / 1e9 / peak if sum(kus) > 0 else None,
                        "cg_solve_ms_same_problem": t, "speedup_vs_cg": t / te}), flush=True)
                    # f3 x f4: BiCGSTAB on the Schur operator (even-odd preconditioned BiCGSTAB)
                    for _ in range(2):
                        ctx.bicgstab_solve_eo(Ue, ee, cfg.kappa, r_min, cfg.max_iter, out=pe)
                    ctx.wd_set_poll_interval(1)     # one sampled iteration per poll chunk: sample them all
                    ctx.wd_set_profile(True)
                    for _ in range(3):
                        ctx.bicgstab_solve_eo(Ue, ee, cfg.kappa, r_min, cfg.max_iter, out=pe)
                    pb = ctx.wd_get_profile_eo_bicgstab()
                    ctx.wd_set_profile(False)
                    ctx.wd_set_poll_interval(0)
                    ms = []
                    for _ in range(5):
                        _, ieb = ctx.bicgstab_solve_eo(Ue, ee, cfg.kappa, r_min, cfg.max_iter, out=pe)
                        ms.append(ieb["gpu_ms"])
                    kus = [m / max(pb["iterations"], 1) * 1e3 for m in pb["ms"]]
                    hb = (sb + gb, 2 * sb + gb, 3 * sb // 2, sb + gb, 3 * sb // 2 + gb, 7 * sb // 2, 2 * sb)
                    teb = float(np.median(ms))
                    names = ("H_oe_p", "M_rv", "s", "H_oe_s", "M_ts", "xr", "p")
                    print(json.dumps({
                        "row": "f3xf4 even-odd bicgstab", "config": ci, "precision": prec, "iterations": ieb["iterations"],
                        "status": ieb["status"], "rel_residual": ieb["rel_residual"], "solve_ms": teb,
                        "kernel_us": dict(zip(names, kus)), "bytes_per_full_site": dict(zip(names, hb)),
                        "kernel_gbs": dict(zip(names, [b * V / (u * 1e-6) / 1e9 if u > 0 else None for b, u in zip(hb, kus)])),
                        "iteration_gbs": sum(hb) * V / (sum(kus) * 1e-6) / 1e9 if sum(kus) > 0 else None,
                        "iteration_frac_of_measured": sum(hb) * V / (sum(kus) * 1e-6) / 1e9 / peak if sum(kus) > 0 else None,
                        "cg_solve_ms_same_problem": t, "speedup_vs_cg": t / teb}), flush=True)
                    # ... and on 12-real links (the two byte reductions of f3 composed with f4)
                    ctx.wd_set_gauge_recon(12)
                    U12 = ctx.wd_eo_pack_gauge(torch.from_numpy(U).cuda())
                    for _ in range(2):
                        ctx.bicgstab_solve_eo(U12, ee, cfg.kappa, r_min, cfg.max_iter, out=pe)
                    ctx.wd_set_poll_interval(1)
                    ctx.wd_set_profile(True)
                    for _ in range(3):
                        ctx.bicgstab_solve_eo(U12, ee, cfg.kappa, r_min, cfg.max_iter, out=pe)
                    pb = ctx.wd_get_profile_eo_bicgstab()
                    ctx.wd_set_profile(False)
                    ctx.wd_set_poll_interval(0)
                    ms = []
                    for _ in range(5):
                        _, ie12 = ctx.bicgstab_solve_eo(U12, ee, cfg.kappa, r_min, cfg.max_iter, out=pe)
                        ms.append(ie12["gpu_ms"])
                    kus = [m / max(pb["iterations"], 1) * 1e3 for m in pb["ms"]]
                    g12 = 48 * rb
                    hb = (sb + g12, 2 * sb + g12, 3 * sb // 2, sb + g12, 3 * sb // 2 + g12, 7 * sb // 2, 2 * sb)
                    t12 = float(np.median(ms))
                    print(json.dumps({
                        "row": "f3xf4 even-odd bicgstab, 12-real links", "config": ci, "precision": prec,
                        "iterations": ie12["iterations"], "status": ie12["status"], "rel_residual": ie12["rel_residual"],
                        "solve_ms": t12, "kernel_us": dict(zip(names, kus)), "bytes_per_full_site": dict(zip(names, hb)),
                        "kernel_gbs": dict(zip(names, [b * V / (u * 1e-6) / 1e9 if u > 0 else None for b, u in zip(hb, kus)])),
                        "iteration_gbs": sum(hb) * V / (sum(kus) * 1e-6) / 1e9 if sum(kus) > 0 else None,
                        "iteration_frac_of_measured": sum(hb) * V / (sum(kus) * 1e-6) / 1e9 / peak if sum(kus) > 0 else None,
                        "cg_solve_ms_same_problem": t, "speedup_vs_cg": t / t12}), flush=True)
                    ctx.wd_set_gauge_recon(18)
                    del Ue, U12, ee, pe
    # f2: the paper's COO SpMV at its largest volume (14^4) and at 32^4 (9.9 GB of Val / Row / Col in fp32)
    for ci in (2, 3):
        run_coo_row(torch, wilson, ci, prec, peak)
    return 0


def run_coo_row(torch, wilson, ci, prec, peak):
    """wd_coo_spmv on the arrays wd_coo_assemble wrote: the sorted-row fast path and, beside it, the any-order atomic
    kernel (wd_set_coo_fast(0)), as GB/s of the algorithmic 9600 B/site (fp32) and as GFLOP/s at 8 flop per entry."""
    cfg = inputs.CONFIGS[ci]
    rb = 4 if prec == 32 else 8
    U, eta = inputs.config_inputs(cfg, dtype=np.complex64 if prec == 32 else np.complex128)
    V = cfg.volume
    with wilson.WilsonContext(cfg.dims, prec, cfg.bc_t) as ctx:
        Un = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
        eta_d = torch.from_numpy(eta).cuda()
        en = ctx.wd_pack_spinor(eta_d)
        out_n = ctx.empty_spinor()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        val, row, col = ctx.wd_coo_assemble(Un, cfg.kappa, False)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(10):
            ctx.lib.wd_coo_assemble(ctx._ctx, ctx._p(Un), cfg.kappa, 0, ctx._p(val), ctx._p(row), ctx._p(col))
        e1.record()
        torch.cuda.synchronize()
        asm_ms = e0.elapsed_time(e1) / 10
        out = torch.empty_like(eta_d)
        reps = 100 if ci == 2 else 20
        times = {}
        for fast in (1, 0):
            ctx.wd_set_coo_fast(fast)
            for _ in range(5):
                ctx.wd_coo_spmv(val, row, col, eta_d, out=out)
            e0.record()
            for _ in range(reps):
                ctx.wd_coo_spmv(val, row, col, eta_d, out=out)
            e1.record()
            torch.cuda.synchronize()
            times[fast] = e0.elapsed_time(e1) / reps
        ctx.wd_set_coo_fast(1)
        st_ms = time_wd_apply(ctx, Un, en, out_n, cfg.kappa, False)
        nnz = NNZ_PER_SITE * V
        coo_bytes = nnz * (2 * rb + 8) + 2 * 12 * V * 2 * rb   # Val + Row + Col once, in and out vectors once
        gbs = lambda ms: coo_bytes / (ms * 1e-3) / 1e9
        print(json.dumps({
            "row": "f2 coo spmv", "config": ci, "name": cfg.name, "precision": prec, "nnz": nnz, "assemble_ms": asm_ms,
            "spmv_us": times[1] * 1e3, "spmv_gflops_8_per_nnz": FLOP_COO_NNZ * nnz / (times[1] * 1e-3) / 1e9,
            "spmv_gbs": gbs(times[1]), "spmv_frac_of_measured": gbs(times[1]) / peak,
            "any_order_kernel_us": times[0] * 1e3, "any_order_kernel_gbs": gbs(times[0]),
            "any_order_kernel_frac_of_measured": gbs(times[0]) / peak,
            "bytes_per_site": coo_bytes / V, "coo_bytes_total": coo_bytes, "stencil_wd_apply_us": st_ms * 1e3,
            "stencil_speedup": times[1] / st_ms,
            "paper": "about 65 GFLOP/s COO SpMV on an A100-PCIE-40GB (PAPER.md:96), other hardware: context only"}), flush=True)


def run_sweep(args, cfg, ctx, wilson, Un, en, psi_n, r_min):
    """Per launch configuration: device time of a2 / a3 / a4 per CG iteration (CUDA events inside the solve) and
    of a standalone wd_apply, as achieved algorithmic GB/s."""
    import torch

    V = cfg.volume
    b2, b3, b4 = (480, 576, 480) if args.precision == 32 else (960, 1152, 960)
    only = [int(t) for t in args.sweep_tiles.split(",")] if args.sweep_tiles else None
    for tile, inf in enumerate(wilson.tile_infos()):
        if only is not None and tile not in only:
            continue
        try:
            ctx.wd_set_tile(tile)
        except wilson.WilsonError:
            continue  # not compiled for this precision
        ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=psi_n)
        ctx.wd_set_profile(True)
        for _ in range(max(1, args.steps)):
            _, info = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=psi_n)
        p = ctx.wd_get_profile()
        ctx.wd_set_profile(False)
        n = max(p["iterations"], 1)
        a2, a3, a4 = p["a2_ms"] / n, p["a3_ms"] / n, p["a4_ms"] / n
        ap_ms = time_wd_apply(ctx, Un, en, psi_n, cfg.kappa, False)
        gbs = lambda b, ms: b * V / (ms * 1e-3) / 1e9 if ms > 0 else None
        print(json.dumps({
            "sweep": f"config{cfg.index}", "precision": args.precision, "tile_index": tile, "tile": list(inf[:4]),
            "threads": inf[0] * inf[1] * inf[2] * inf[3], "min_blocks_per_sm": inf[4], "has_fp32": inf[5],
            "iterations": info["iterations"], "a2_us": a2 * 1e3, "a3_us": a3 * 1e3, "a4_us": a4 * 1e3,
            "a2_gbs": gbs(b2, a2), "a3_gbs": gbs(b3, a3), "a4_gbs": gbs(b4, a4),
            "cg_iteration_gbs": gbs(b2 + b3 + b4, a2 + a3 + a4), "solve_ms": info["gpu_ms"],
            "wd_apply_x100_us": ap_ms * 1e3, "wd_apply_gbs": gbs(b2, ap_ms),
            "wd_apply_gflops": FLOP_APPLY * V / (ap_ms * 1e-3) / 1e9}), flush=True)
    ctx.close()
    return 0


def run_staging(args):
    """Per row of the staged stencil (and -1 = links through L1, first and last): a2 / a3 / a4 per CG iteration from CUDA
    events inside `--steps` solves, the solve time, wd_apply over `--reps` applications, and whether wd_apply is
    bit-identical to the unstaged kernel."""
    import torch

    from . import build as wbuild
    from . import wilson

    wbuild.build()
    wilson.load_library()
    prec = args.precision
    cfg = inputs.CONFIGS[args.config]
    r_min = cfg.r_min if prec == 32 else 1e-10
    U, eta = inputs.config_inputs(cfg, dtype=np.complex64 if prec == 32 else np.complex128)
    V = cfg.volume
    b2, b3, b4 = (480, 576, 480) if prec == 32 else (960, 1152, 960)
    with wilson.WilsonContext(cfg.dims, prec, cfg.bc_t) as ctx:
        ctx.wd_set_cg_mode(1)
        Un = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
        en = ctx.wd_pack_spinor(torch.from_numpy(eta).cuda())
        out = ctx.empty_spinor()
        infos = wilson.staging_rows()
        rows = [i for i, inf in enumerate(infos) if inf[7 if prec == 32 else 8] and all(cfg.dims[d] % inf[d] == 0 for d in range(4))]
        if args.staging_rows:
            rows = [r for r in rows if r in [int(v) for v in args.staging_rows.split(",")]]
        ref = None
        for row in [-1] + rows + [-1]:
            ctx.wd_set_link_staging(row)
            if args.steps > 0:
                ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
                ctx.wd_set_profile(1)
                ms = []
                for _ in range(args.steps):
                    _, info = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
                    ms.append(info["gpu_ms"])
                p = ctx.wd_get_profile()
                ctx.wd_set_profile(0)
            else:
                p, ms, info = {"a2_ms": 0.0, "a3_ms": 0.0, "a4_ms": 0.0, "iterations": 0}, [0.0], {"iterations": 0}
            n = max(p["iterations"], 1)
            ap = sorted(ctx.wd_apply_repeat(Un, en, cfg.kappa, True, args.reps, out=out) for _ in range(3))[1]
            got = out.clone()
            ref = got if ref is None else ref
            a2, a3, a4 = p["a2_ms"] / n, p["a3_ms"] / n, p["a4_ms"] / n
            gbs = lambda b, t: b * V / (t * 1e-3) / 1e9 if t > 0 else None
            print(json.dumps({
                "staging": f"config{cfg.index}", "precision": prec, "row": row,
                "tile_stages_buffers_minb": list(infos[row][:7]) if row >= 0 else None,
                "a2_us": a2 * 1e3, "a3_us": a3 * 1e3, "a4_us": a4 * 1e3, "a2_gbs": gbs(b2, a2), "a3_gbs": gbs(b3, a3),
                "cg_iteration_gbs": gbs(b2 + b3 + b4, a2 + a3 + a4), "solve_ms": float(np.median(ms)),
                "iterations": info["iterations"], "wd_apply_dagger_us": ap * 1e3, "wd_apply_gbs": gbs(b2, ap),
                "bit_identical_to_unstaged": bool(torch.equal(got, ref))}), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--report", action="store_true")
    ap.add_argument("--rows", action="store_true")
    ap.add_argument("--rows-configs", default="3,4", help="configs the solver rows of --rows run on (comma separated)")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--sweep-tiles", default="", help="launch configurations --sweep visits (comma separated; default all)")
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--precision", type=int, default=32, choices=[32, 64])
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--coo", action="store_true", help="only the COO SpMV rows of --rows (14^4 and 32^4)")
    ap.add_argument("--staging", action="store_true")
    ap.add_argument("--staging-rows", default="", help="rows --staging visits (comma separated; default: all that cover the lattice)")
    ap.add_argument("--reps", type=int, default=50, help="wd_apply applications per timing of --staging")
    args = ap.parse_args()
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("measure.py needs a CUDA device: the product path has no CPU fallback")
    if args.report:
        return run_report(args)
    if args.rows:
        return run_rows(args)
    if args.coo:
        from . import build as wbuild
        from . import wilson

        wbuild.build()
        wilson.load_library()
        for ci in (2, 3):
            run_coo_row(torch, wilson, ci, args.precision, measured_peak()[0])
        return 0
    if args.staging:
        return run_staging(args)
    if args.sweep:
        from . import build as wbuild
        from . import wilson

        wbuild.build()
        wilson.load_library()
        cfg = inputs.CONFIGS[args.config]
        r_min = cfg.r_min if args.precision == 32 else 1e-10
        U, eta = inputs.config_inputs(cfg, dtype=np.complex64 if args.precision == 32 else np.complex128)
        ctx = wilson.WilsonContext(cfg.dims, args.precision, cfg.bc_t)
        Un = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
        en = ctx.wd_pack_spinor(torch.from_numpy(eta).cuda())
        return run_sweep(args, cfg, ctx, wilson, Un, en, ctx.empty_spinor(), r_min)
    ap.print_help()
    return 2


if __name__ == "__main__":
    sys.exit(main())
