#!/usr/bin/env python
"""bench.py — the measurement contract of this repo.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--precision 32|64] [--impl ours|reference]
    python bench.py --report | --rows | --sweep        (measurement tables of BASELINE.md; not the bench line)

One "step" = one pass of the whole hot path over one synthetic lattice: cg_solve (a1 init, the fused CG
loop a2-a5 until |r|/|eta| < r_min, a6 final D-dagger) on BASELINE.json's config I (default 4: 48^3x96,
the paper's quoted production volume, and the largest single-GPU config).  The metric is
BASELINE.json's: Wilson D D-dagger CG GFLOP/s with the fixed flop convention (2976 flop/site/iteration +
1368 flop/site for the final D-dagger), plus the achieved fraction of the HBM roofline of the dominant
kernel.  Inputs are seeded and synthetic (paper_2111_14958_b200/inputs.py); they stand in for the paper's
unspecified gauge fields.

`value`   : device-resident inputs (native layout already in HBM), CUDA events around K steps.
`e2e`     : the same solve through the C-ABI host-buffer call cg_solve_host (pinned HOST canonical
            buffers; H2D copies of U and eta, pack, solve, unpack and the D2H copy of psi inside the timed region).
`roofline`: the dominant kernel (a3: D pass + fused r update + |r|^2, 576 B/site fp32) timed live with CUDA
            events around its launches (every 4th iteration) inside the timed steps (wd_set_profile).
`cpu_baseline`: the fp64 CPU oracle, as it stands, on a bounded sample (max_iter = 2) of the same workload.

N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -> N independent replicas
("replicas only"); value = total flops of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2111_14958_b200 import inputs  # noqa: E402

FLOP_ITER = 2976        # per site per CG iteration (reading G14)
FLOP_APPLY = 1368       # per site per D / D-dagger application
BYTES_A3 = {32: 576, 64: 1152}     # a3: read q, U, r; write r
BYTES_ITER = {32: 1536, 64: 3072}  # a2 + a3 + a4
METRIC = "Wilson DD-dagger CG GFLOP/s (fp32, 1 B200; roofline = achieved HBM GB/s fraction)"


def cg_flops(volume, iterations):
    return float(volume) * (FLOP_ITER * iterations + FLOP_APPLY)


def workload_name(cfg, r_min):
    return (f"config{cfg.index}: {cfg.name} Wilson CG on D D-dagger, kappa={cfg.kappa}, links={cfg.links}, "
            f"r_min={r_min:g}, antiperiodic t")


def max_over_ranks(x, dist=None, device="cpu"):
    """Time-like quantity -> max over all ranks (the slowest rank bounds the job).  dist = torch.distributed or None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(x)
    import torch

    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, volume, iterations, seconds):
    """Replicas only: every rank solves the same lattice, so the job's flops are world x one solve; the time is
    the max over ranks."""
    return world * cg_flops(volume, iterations) / seconds / 1e9


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def stored_traffic(cfg_index, precision):
    """dram bytes per launch of the a3 kernel from the committed ncu --set full capture, or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return json.load(f).get(f"config{cfg_index}_fp{precision}_a3")
    except Exception:
        return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML every 100 ms while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None

    def run(self):
        try:
            import pynvml as nv

            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
                getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
            }
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                    for bit, name in names.items():
                        if mask & bit:
                            self.reasons.add(name)
                except Exception:
                    pass
                time.sleep(0.1)
        except Exception as e:  # NVML missing: report that rather than fail the bench
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def result(self):
        self.stop_flag = True
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_sample(cfg, precision, U, eta, sample_iters):
    """The oracle, as it stands, on a bounded sample: `sample_iters` CG iterations + the final D-dagger."""
    from oracle import wilson_oracle

    U64 = U.astype(np.complex128)
    eta64 = eta.astype(np.complex128)
    t0 = time.perf_counter()
    _, info = wilson_oracle.cg_solve(cfg.dims, U64, eta64, cfg.kappa, 1e-30, sample_iters, cfg.bc_t)
    dt = time.perf_counter() - t0
    gflops = cg_flops(cfg.volume, info["iterations"]) / dt / 1e9
    return gflops, dt, wilson_oracle.num_threads(), info["iterations"]


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    sample_iters = args.sample_iters
    U, eta = inputs.config_inputs(cfg, dtype=np.complex64 if args.precision == 32 else np.complex128)
    times, cores, its = [], 1, sample_iters
    for i in range(args.warmup + args.steps):
        gf, dt, cores, its = oracle_sample(cfg, args.precision, U, eta, sample_iters)
        if i >= args.warmup:
            times.append(dt)
    t = float(np.mean(times))
    value = cg_flops(cfg.volume, its) / t / 1e9
    sample = f"{its} CG iterations + final D-dagger of config {cfg.index} ({cfg.name}), fp64 oracle, full lattice"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, cfg.r_min if args.precision == 32 else 1e-10), "volume": cfg.volume,
                   "sample_cg_iterations": its, "parallelism": "host cores (oracle)"},
        "cpu_baseline": {"value": value, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def time_wd_apply(ctx, Un, en, out, kappa, dagger, reps=100):
    """device time per application over `reps` back-to-back applications (enqueued from C by wd_apply_repeat, CUDA
    events on the ctx stream; median of three rounds)"""
    return sorted(ctx.wd_apply_repeat(Un, en, kappa, dagger, reps, out=out) for _ in range(3))[1]


def run_report(args):
    """every config, wd_apply D and D-dagger (100 applications each, BASELINE.json configs[2])
    and the whole CG solve."""
    import torch

    from paper_2111_14958_b200 import build as wbuild
    from paper_2111_14958_b200 import wilson

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


def run_oracle_report(args):
    """SURVEY.md 8(d) "Oracle timing": the fp64 CPU oracle as it stands on this box's host cores, at all cores and at
    one thread.  Full CG at configs 0-2 (both thread counts) and at config 3 (all cores; one thread: 2 iterations);
    config 4: 10 iterations + final D-dagger at all cores, one wd_apply at both thread counts.  One JSON line each.
    Needs no GPU.  Reported baseline, not a target."""
    from oracle import wilson_oracle

    cpu = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            cpu = next(l.split(":", 1)[1].strip() for l in f if l.startswith("model name"))
    except Exception:
        pass
    all_threads = wilson_oracle.num_threads()
    for ci in [int(x) for x in args.rows_configs.split(",") if x] if args.rows_configs != "3,4" else range(5):
        cfg = inputs.CONFIGS[ci]
        U, eta = inputs.config_inputs(cfg, dtype=np.complex64)
        U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
        del U, eta
        V = cfg.volume
        for nt in (all_threads, 1):
            wilson_oracle.set_num_threads(nt)
            reps = max(1, min(100, int(2.0e6 * nt / V)))
            if V <= 1 << 20:
                wilson_oracle.wd_apply(cfg.dims, U64, eta64, cfg.kappa, False, cfg.bc_t)   # warm-up (thread pool start)
            t0 = time.perf_counter()
            for _ in range(reps):
                wilson_oracle.wd_apply(cfg.dims, U64, eta64, cfg.kappa, False, cfg.bc_t)
            apply_s = (time.perf_counter() - t0) / reps
            line = {"oracle_report": f"config{ci}", "name": cfg.name, "volume": V, "threads": nt, "host_cores": os.cpu_count(),
                    "cpu": cpu, "wd_apply_ms": apply_s * 1e3, "wd_apply_gflops": FLOP_APPLY * V / apply_s / 1e9,
                    "wd_apply_applications": reps}
            full = ci <= 2 or (ci == 3 and nt == all_threads)
            iters = cfg.max_iter if full else (10 if (ci == 4 and nt == all_threads) else (2 if ci == 3 else 0))
            if iters:
                t0 = time.perf_counter()
                _, info = wilson_oracle.cg_solve(cfg.dims, U64, eta64, cfg.kappa, cfg.r_min if full else 1e-30, iters, cfg.bc_t)
                dt = time.perf_counter() - t0
                line.update({"cg": "full solve" if full else f"{iters} iterations + final D-dagger",
                             "cg_iterations": info["iterations"], "cg_seconds": dt,
                             "cg_seconds_per_iteration": dt / max(info["iterations"], 1),
                             "cg_gflops": cg_flops(V, info["iterations"]) / dt / 1e9})
            print(json.dumps(line), flush=True)
        wilson_oracle.set_num_threads(all_threads)
    return 0


FLOP_BICG_ITER = 2 * 1368 + 960   # two D applications + 10 complex vector/dot operations
BYTES_BICG = {32: (576, 288, 480, 672, 384), 64: (1152, 576, 960, 1344, 768)}   # the five kernels of one iteration
FLOP_COO_NNZ = 8                   # one complex multiply-add per stored entry
NNZ_PER_SITE = 588


def run_rows(args):
    """The SURVEY.md 8(f) rows, one JSON line each: BiCGSTAB (f4) and 12-real links (f3) at configs 3 and 4, the paper's
    COO SpMV (f2) at 14^4 (config 2, the largest volume of the paper's range) beside the matrix-free stencil."""
    import torch

    from paper_2111_14958_b200 import build as wbuild
    from paper_2111_14958_b200 import wilson

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
                print(json.dumps({
                    "row": "f3 link storage", "config": ci, "precision": prec, "reals_per_link": recon,
                    "bytes_per_site": {"wd_apply": b2, "a2": b2, "a3": b3, "a4": b4, "cg_iteration": b2 + b3 + b4},
                    "wd_apply_D_us": d_ms * 1e3, "wd_apply_D_gbs": b2 * V / (d_ms * 1e-3) / 1e9,
                    "cg_iterations": info["iterations"], "cg_solve_ms": t,
                    "cg_gflops": cg_flops(V, info["iterations"]) / (t * 1e-3) / 1e9,
                    "a2_us": a2 * 1e3, "a3_us": a3 * 1e3, "a4_us": a4 * 1e3,
                    "a2_gbs": b2 * V / (a2 * 1e-3) / 1e9, "a3_gbs": b3 * V / (a3 * 1e-3) / 1e9,
                    "cg_iteration_gbs": (b2 + b3 + b4) * V / ((a2 + a3 + a4) * 1e-3) / 1e9,
                    "cg_iteration_frac_of_measured": (b2 + b3 + b4) * V / ((a2 + a3 + a4) * 1e-3) / 1e9 / peak}), flush=True)
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
    # f2: the paper's COO SpMV at its largest volume
    cfg = inputs.CONFIGS[2]
    U, eta = inputs.config_inputs(cfg, dtype=cdt)
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
        for _ in range(5):
            ctx.wd_coo_spmv(val, row, col, eta_d, out=out)
        reps = 100
        e0.record()
        for _ in range(reps):
            ctx.wd_coo_spmv(val, row, col, eta_d, out=out)
        e1.record()
        torch.cuda.synchronize()
        sp_ms = e0.elapsed_time(e1) / reps
        st_ms = time_wd_apply(ctx, Un, en, out_n, cfg.kappa, False)
        nnz = NNZ_PER_SITE * V
        coo_bytes = nnz * (2 * rb + 8) + 2 * 12 * V * 2 * rb   # Val + Row + Col once, in and out vectors once
        print(json.dumps({
            "row": "f2 coo spmv", "config": 2, "precision": prec, "nnz": nnz, "assemble_ms": asm_ms,
            "spmv_us": sp_ms * 1e3, "spmv_gflops_8_per_nnz": FLOP_COO_NNZ * nnz / (sp_ms * 1e-3) / 1e9,
            "spmv_gbs": coo_bytes / (sp_ms * 1e-3) / 1e9, "spmv_frac_of_measured": coo_bytes / (sp_ms * 1e-3) / 1e9 / peak,
            "bytes_per_site": coo_bytes / V, "stencil_wd_apply_us": st_ms * 1e3,
            "stencil_speedup": sp_ms / st_ms,
            "paper": "about 65 GFLOP/s COO SpMV on an A100-PCIE-40GB (PAPER.md:96), other hardware: context only"}), flush=True)
    return 0


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
            "threads": inf[0] * inf[1] * inf[2] * inf[3], "min_blocks_per_sm": inf[4], "pipeline": inf[5],
            "iterations": info["iterations"], "a2_us": a2 * 1e3, "a3_us": a3 * 1e3, "a4_us": a4 * 1e3,
            "a2_gbs": gbs(b2, a2), "a3_gbs": gbs(b3, a3), "a4_gbs": gbs(b4, a4),
            "cg_iteration_gbs": gbs(b2 + b3 + b4, a2 + a3 + a4), "solve_ms": info["gpu_ms"],
            "wd_apply_x100_us": ap_ms * 1e3, "wd_apply_gbs": gbs(b2, ap_ms),
            "wd_apply_gflops": FLOP_APPLY * V / (ap_ms * 1e-3) / 1e9}), flush=True)
    ctx.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index (default 4: 48^3x96)")
    ap.add_argument("--precision", type=int, default=32, choices=[32, 64])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--tile", type=int, default=-1, help="CTA tile index (-1 = library's automatic choice)")
    ap.add_argument("--sample-iters", type=int, default=2, help="CG iterations of the oracle's bounded sample")
    ap.add_argument("--sweep", action="store_true",
                    help="time every compiled launch configuration (the paper's workgroup-size tuning, PAPER.md:76) "
                         "on this config and print one JSON line per configuration instead of the bench line")
    ap.add_argument("--sweep-tiles", default="", help="launch configurations --sweep visits (comma separated; default all)")
    ap.add_argument("--report", action="store_true",
                    help="one JSON line per BASELINE config (0..4, plus config 3 in fp64): wd_apply D / D-dagger over 100 "
                         "applications and the CG solve; the table of BASELINE.md section 3")
    ap.add_argument("--rows", action="store_true",
                    help="one JSON line per SURVEY.md 8(f) row: 12-real links and BiCGSTAB at configs 3 and 4, the paper's COO "
                         "SpMV at 14^4 beside the stencil")
    ap.add_argument("--rows-configs", default="3,4", help="configs the solver rows of --rows run on (comma separated)")
    ap.add_argument("--oracle-report", action="store_true",
                    help="time the fp64 CPU oracle on this box's host cores at all cores and at one thread (SURVEY.md 8(d)); "
                         "needs no GPU; --rows-configs selects the configs (default all five)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    cfg = inputs.CONFIGS[args.config]
    r_min = cfg.r_min if args.precision == 32 else 1e-10
    if args.impl == "reference":
        return run_reference(args, cfg)
    if args.oracle_report:
        return run_oracle_report(args) if int(os.environ.get("RANK", "0")) == 0 else 0

    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if args.report:
        return run_report(args) if rank == 0 else 0
    if args.rows:
        return run_rows(args) if rank == 0 else 0
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2111_14958_b200 import build as wbuild
    from paper_2111_14958_b200 import wilson

    if rank == 0:
        wbuild.build()
    if dist:
        dist.barrier()
    wilson.load_library()

    cdt = np.complex64 if args.precision == 32 else np.complex128
    U, eta = inputs.config_inputs(cfg, dtype=cdt)   # seeded, identical on every rank (replicas)
    V = cfg.volume
    ctx = wilson.WilsonContext(cfg.dims, args.precision, cfg.bc_t)
    if args.tile >= 0:
        ctx.wd_set_tile(args.tile)
    U_dev = torch.from_numpy(U).cuda()
    Un = ctx.wd_pack_gauge(U_dev)
    del U_dev
    eta_dev = torch.from_numpy(eta).cuda()
    en = ctx.wd_pack_spinor(eta_dev)
    del eta_dev
    psi_n = ctx.empty_spinor()
    torch.cuda.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
            torch.cuda.synchronize()

    if args.sweep:
        return run_sweep(args, cfg, ctx, wilson, Un, en, psi_n, r_min)

    # ---------------- device-resident arm
    for _ in range(args.warmup):
        ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=psi_n)
    # CUDA events around the three kernels of every 4th iteration of the timed solves (31 of 124 iterations per solve at
    # config 4): every launch costs about 1.5 us of stream time per event, which is 2 % of an iteration at 32^4
    ctx.wd_set_profile(4)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches, iters = 0, 0
    e0.record()
    for _ in range(args.steps):
        _, info = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=psi_n)
        launches += info["kernel_launches"]
        iters = info["iterations"]
    e1.record()
    barrier()
    clocks = sampler.result()
    ms_total = e0.elapsed_time(e1)
    prof = ctx.wd_get_profile()
    ctx.wd_set_profile(False)
    ms_total = max_over_ranks(ms_total, dist, "cuda")
    ms_step = ms_total / args.steps
    value = whole_job_value(world, V, iters, ms_step * 1e-3)

    # ---------------- roofline of the dominant kernel (a3), timed live inside the steps above
    peak, peak_src = measured_peak()
    a3_ms = prof["a3_ms"] / max(prof["iterations"], 1)
    a3_bytes = BYTES_A3[args.precision] * V
    achieved = a3_bytes / (a3_ms * 1e-3) / 1e9 if a3_ms > 0 else None
    iter_ms = (prof["a2_ms"] + prof["a3_ms"] + prof["a4_ms"]) / max(prof["iterations"], 1)
    roofline = {
        "bound": "hbm", "kernel": "dslash_kernel<MODE_RUPD> (a3: D pass + r update + |r|^2)",
        "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak if achieved else None,
        "peak_source": peak_src, "traffic": stored_traffic(cfg.index, args.precision),
        "algorithmic_bytes_per_launch": a3_bytes, "avg_launch_ms": a3_ms,
        "per_kernel_ms": {"a2": prof["a2_ms"] / max(prof["iterations"], 1), "a3": a3_ms,
                          "a4": prof["a4_ms"] / max(prof["iterations"], 1)},
        "cg_iteration": {"achieved": BYTES_ITER[args.precision] * V / (iter_ms * 1e-3) / 1e9 if iter_ms > 0 else None,
                         "frac": BYTES_ITER[args.precision] * V / (iter_ms * 1e-3) / 1e9 / peak if iter_ms > 0 else None,
                         "frac_of_8TBs": BYTES_ITER[args.precision] * V / (iter_ms * 1e-3) / 1e9 / 8000.0 if iter_ms > 0 else None,
                         "bytes_per_site": BYTES_ITER[args.precision], "ms": iter_ms},
    }

    # ---------------- end to end through the host-buffer C-ABI call
    e2e = None
    if not args.no_e2e:
        U_pin = torch.from_numpy(U).pin_memory()
        eta_pin = torch.from_numpy(eta).pin_memory()
        psi_pin = torch.empty((V, 4, 3), dtype=torch.complex64 if args.precision == 32 else torch.complex128).pin_memory()
        ctx.cg_solve_host(U_pin, eta_pin, cfg.kappa, r_min, cfg.max_iter, out=psi_pin)  # warm-up (allocates staging)
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 3))
        for _ in range(n_e2e):
            _, info_h = ctx.cg_solve_host(U_pin, eta_pin, cfg.kappa, r_min, cfg.max_iter, out=psi_pin)
        barrier()
        dt = (time.perf_counter() - t0) / n_e2e
        dt = max_over_ranks(dt, dist, "cuda")
        e2e = {"value": whole_job_value(world, V, info_h["iterations"], dt), "unit": "GFLOP/s",
               "h2d_bytes_per_step": int(U.nbytes + eta.nbytes), "d2h_bytes_per_step": int(eta.nbytes),
               "ms_per_step": dt * 1e3, "steps": n_e2e}
        del U_pin, eta_pin, psi_pin

    # ---------------- the oracle on the host cores (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        gf, dt, cores, its = oracle_sample(cfg, args.precision, U, eta, args.sample_iters)
        cpu = {"value": gf, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": f"{its} CG iterations + final D-dagger of config {cfg.index} ({cfg.name}), fp64 oracle, full lattice"}

    ws_bytes = (72 + 24 * 6) * V * (4 if args.precision == 32 else 8)
    line = {
        "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if args.precision == 32 else "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, r_min), "volume": V, "cg_iterations": iters, "tile": list(wilson.tile_shapes()[ctx.wd_get_tile()]),
                   "l2_policy": f"inputs larger than L2 (working set {ws_bytes / 1e6:.0f} MB vs 126 MB L2)"
                   if ws_bytes > 2 * 126e6 else "working set fits L2 (latency-bound regime, no roofline claim)",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
    }
    if rank == 0:
        print(json.dumps(line), flush=True)
    ctx.close()
    if dist:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
