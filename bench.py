#!/usr/bin/env python
"""bench.py — the measurement contract of this repo.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--precision 32|64] [--impl ours|reference]
(the measurement tables of BASELINE.md come from `python -m paper_2111_14958_b200.measure --report | --rows | --sweep`)

One "step" = one pass of the whole hot path over one synthetic lattice: cg_solve (a1 init, the fused CG
loop a2-a5 until |r|/|eta| < r_min, a6 final D-dagger) on BASELINE.json's config I (default 4: 48^3x96,
the paper's quoted production volume, and the largest single-GPU config).  The metric is
BASELINE.json's: Wilson D D-dagger CG GFLOP/s with the fixed flop convention (2976 flop/site/iteration +
1368 flop/site for the final D-dagger), plus the achieved fraction of the HBM roofline of the dominant
kernel.  Inputs are seeded and synthetic (paper_2111_14958_b200/inputs.py); they stand in for the paper's
unspecified gauge fields.

`value`   : device-resident inputs (native layout already in HBM), CUDA events around K steps.
`e2e`     : the same solves through the C-ABI host-buffer calls (pinned HOST canonical buffers; per step the H2D copies
            of U and eta, pack, solve, unpack and the D2H copy of psi, all inside the timed region).  `value` = the K
            steps as a queue pipelined over two contexts (cg_solve_host_begin / _run / _wait: the transfers of one step
            overlap the iterations of its neighbours); `one_call_at_a_time` = the same K steps as K cg_solve_host calls.
`roofline`: the dominant kernel (a3: D pass + fused r update + |r|^2, 576 B/site fp32) timed live with CUDA
            events around its launches (every 4th iteration) inside the timed steps (wd_set_profile);
            `roofline.kernels` lists a2, a3, a4 the same way and `roofline.cg_iteration` the fused iteration
            (1536 B/site fp32), the quantity BASELINE.json's target (>= 70 % of the HBM roofline) is stated on.
`also`    : the same device-resident measurement at 32^4 in fp32 and fp64 (BASELINE.json configs[3]: the other
            half of the target statement), a few seconds after the headline solve; only on the default workload.
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


BYTES_A2 = {32: 480, 64: 960}      # a2: read p, U; write q
BYTES_A4 = {32: 480, 64: 960}      # a4: read y, p, r; write y, p


def kernel_table(prof, precision, volume, peak):
    """a2 / a3 / a4 from the CUDA events cg_solve recorded around its launches: algorithmic bytes per launch (SURVEY.md
    8(d) bytes per site x sites), average launch time, achieved GB/s and its fraction of the measured copy peak."""
    n = max(prof["iterations"], 1)
    rows = []
    for name, key, bps in (("a2 dslash_kernel<MODE_QQ>: D-dagger pass + |q|^2", "a2_ms", BYTES_A2[precision]),
                           ("a3 dslash_kernel<MODE_RUPD>: D pass + r update + |r|^2", "a3_ms", BYTES_A3[precision]),
                           ("a4 cg_update_kernel: y += alpha p, p = r + beta p", "a4_ms", BYTES_A4[precision])):
        ms = prof[key] / n
        ach = bps * volume / (ms * 1e-3) / 1e9 if ms > 0 else None
        rows.append({"name": name, "bytes_per_launch": bps * volume, "avg_ms": ms, "achieved": ach,
                     "frac": ach / peak if ach else None, "launches_timed": prof["iterations"]})
    it_ms = sum(r["avg_ms"] for r in rows)
    it_gbs = BYTES_ITER[precision] * volume / (it_ms * 1e-3) / 1e9 if it_ms > 0 else None
    iteration = {"achieved": it_gbs, "frac": it_gbs / peak if it_gbs else None,
                 "frac_of_8TBs": it_gbs / 8000.0 if it_gbs else None, "bytes_per_site": BYTES_ITER[precision], "ms": it_ms}
    return rows, iteration


def time_device_resident(torch, wilson, cfg, precision, steps, warmup, local, dist, world, tile=-1, keep=False):
    """W warm-up solves, then K timed cg_solve calls on inputs already packed in HBM (CUDA events on the ctx stream =
    torch's current stream, barrier + synchronize on both sides, max over ranks), NVML clocks sampled during the timed
    region, per-kernel events on every 4th iteration."""
    cdt = np.complex64 if precision == 32 else np.complex128
    r_min = cfg.r_min if precision == 32 else 1e-10
    U, eta = inputs.config_inputs(cfg, dtype=cdt)   # seeded, identical on every rank (replicas)
    V = cfg.volume
    ctx = wilson.WilsonContext(cfg.dims, precision, cfg.bc_t)
    if tile >= 0:
        ctx.wd_set_tile(tile)
    U_dev = torch.from_numpy(U).cuda()
    Un = ctx.wd_pack_gauge(U_dev)
    del U_dev
    eta_dev = torch.from_numpy(eta).cuda()
    en = ctx.wd_pack_spinor(eta_dev)
    del eta_dev
    psi_n = ctx.empty_spinor()

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(warmup):
        ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=psi_n)
    # CUDA events around the three kernels of every 4th iteration of the timed solves (31 of 124 iterations per solve at
    # config 4): every event costs about 1.5 us of stream time, which is 2 % of an iteration at 32^4
    ctx.wd_set_profile(4)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches, iters = 0, 0
    e0.record()
    for _ in range(steps):
        _, info = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=psi_n)
        launches += info["kernel_launches"]
        iters = info["iterations"]
    e1.record()
    barrier()
    clocks = sampler.result()
    ms_step = max_over_ranks(e0.elapsed_time(e1), dist, "cuda") / steps
    prof = ctx.wd_get_profile()
    ctx.wd_set_profile(False)
    out = {"cfg": cfg, "precision": precision, "r_min": r_min, "V": V, "iters": iters, "launches": launches,
           "ms_step": ms_step, "value": whole_job_value(world, V, iters, ms_step * 1e-3), "clocks": clocks, "prof": prof,
           "tile": list(wilson.tile_shapes()[ctx.wd_get_tile()]), "cg_mode": info["cg_mode"], "status": info["status"]}
    if keep:
        out.update({"ctx": ctx, "U": U, "eta": eta, "barrier": barrier})
    else:
        ctx.close()
        del Un, en, psi_n
        torch.cuda.empty_cache()
    return out


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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the 32^4 fp32 / fp64 measurements after the headline")
    args = ap.parse_args()
    cfg = inputs.CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
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
    peak, peak_src = measured_peak()

    # ---------------- device-resident arm (the headline workload)
    m = time_device_resident(torch, wilson, cfg, args.precision, args.steps, args.warmup, local, dist, world, args.tile,
                             keep=True)
    ctx, U, eta, barrier, V, r_min = m["ctx"], m["U"], m["eta"], m["barrier"], m["V"], m["r_min"]

    # ---------------- roofline of the dominant kernel (a3), timed live inside the steps above
    kernels, iteration = kernel_table(m["prof"], args.precision, V, peak)
    a3 = kernels[1]
    roofline = {
        "bound": "hbm", "kernel": "dslash_kernel<MODE_RUPD> (a3: D pass + r update + |r|^2)",
        "achieved": a3["achieved"], "peak": peak, "unit": "GB/s", "frac": a3["frac"],
        "peak_source": peak_src, "traffic": stored_traffic(cfg.index, args.precision),
        "algorithmic_bytes_per_launch": a3["bytes_per_launch"], "avg_launch_ms": a3["avg_ms"],
        "kernels": kernels, "cg_iteration": iteration,
    }

    # ---------------- end to end through the host-buffer C-ABI call (same number of steps as `value`)
    e2e = None
    if not args.no_e2e:
        U_pin = torch.from_numpy(U).pin_memory()
        eta_pin = torch.from_numpy(eta).pin_memory()
        psi_pin = torch.empty((V, 4, 3), dtype=torch.complex64 if args.precision == 32 else torch.complex128).pin_memory()
        ctx.cg_solve_host(U_pin, eta_pin, cfg.kappa, r_min, cfg.max_iter, out=psi_pin)  # warm-up (allocates staging)
        # what this box's PCIe link gives a plain pinned copy of the same buffers (H2D U + eta, then D2H psi): the
        # floor of the host-buffer form, since the solve needs all of U and eta before its first iteration
        dev_buf = torch.empty_like(U_pin, device="cuda")
        dev_s = torch.empty_like(eta_pin, device="cuda")
        barrier()
        t0 = time.perf_counter()
        dev_buf.copy_(U_pin, non_blocking=True)
        dev_s.copy_(eta_pin, non_blocking=True)
        psi_pin.copy_(dev_s, non_blocking=True)
        torch.cuda.synchronize()
        plain_copy_ms = (time.perf_counter() - t0) * 1e3
        del dev_buf, dev_s
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            _, info_h = ctx.cg_solve_host(U_pin, eta_pin, cfg.kappa, r_min, cfg.max_iter, out=psi_pin)
        barrier()
        dt = (time.perf_counter() - t0) / args.steps
        dt = max_over_ranks(dt, dist, "cuda")
        h2d, d2h = int(U.nbytes + eta.nbytes), int(eta.nbytes)
        e2e = {"value": whole_job_value(world, V, info_h["iterations"], dt), "unit": "GFLOP/s",
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": dt * 1e3, "steps": args.steps,
               # gpu_ms = the solve itself inside the last host-buffer call (CUDA events around cg_device); the rest of the
               # step is transfers (+ the pack / unpack kernels that do not hide behind them)
               "device_solve_ms_inside": info_h["gpu_ms"], "transfer_ms": dt * 1e3 - info_h["gpu_ms"],
               "effective_pcie_gbs": (h2d + d2h) / max(dt - info_h["gpu_ms"] * 1e-3, 1e-9) / 1e9,
               "plain_pinned_copy_ms_same_bytes": plain_copy_ms, "plain_pinned_copy_gbs": (h2d + d2h) / plain_copy_ms / 1e6}
        # The same K solves as a QUEUE: two contexts on two streams, split-phase calls (cg_solve_host_begin / _run / _wait).
        # Every step still uploads its own U and eta from pinned memory and downloads its own psi inside the timed region;
        # the uploads of step i+1 and the download of step i-1 run while the GPU iterates on step i.  Pipeline fill (the
        # first upload) and drain (the last download) are inside the timed region too.
        psi_pin2 = torch.empty_like(psi_pin).pin_memory()
        # streams above the lowest priority: the library's pack kernels run on a lowest-priority stream of their own and
        # take only the room the other context's solve leaves
        streams = [torch.cuda.Stream(priority=-1), torch.cuda.Stream(priority=-1)]
        pctx = [wilson.WilsonContext(cfg.dims, args.precision, cfg.bc_t, stream=st) for st in streams]
        for pc in pctx:
            if args.tile is not None:
                pc.wd_set_tile(args.tile)
        outs = [psi_pin, psi_pin2]

        def pipelined(nsteps):
            return wilson.cg_solve_host_queue(pctx, [(U_pin, eta_pin)] * nsteps, cfg.kappa, r_min, cfg.max_iter,
                                              [outs[i % 2] for i in range(nsteps)])[-1]

        pipelined(2)                                    # warm-up: staging buffers of both contexts
        barrier()
        t0 = time.perf_counter()
        info_p = pipelined(args.steps)
        barrier()
        dtp = max_over_ranks((time.perf_counter() - t0) / args.steps, dist, "cuda")
        same = bool(torch.equal(psi_pin, psi_pin2)) if args.steps > 1 else None
        for pc in pctx:
            pc.close()
        serial = {k: e2e[k] for k in ("value", "ms_per_step", "device_solve_ms_inside", "transfer_ms", "effective_pcie_gbs")}
        e2e.update({"value": whole_job_value(world, V, info_p["iterations"], dtp), "ms_per_step": dtp * 1e3,
                    "mode": "queue of K solves pipelined over 2 contexts / streams (cg_solve_host_begin, _run, _wait): every "
                            "step copies its own inputs H2D and its result D2H inside the timed region, overlapped with the "
                            "neighbouring steps' iterations; fill and drain included",
                    "device_solve_ms_inside": info_p["gpu_ms"], "outputs_identical": same,
                    "one_call_at_a_time": serial})
        del e2e["transfer_ms"], e2e["effective_pcie_gbs"]
        del U_pin, eta_pin, psi_pin, psi_pin2
    ctx.close()
    torch.cuda.empty_cache()

    # ---------------- the oracle on the host cores (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        gf, dt, cores, its = oracle_sample(cfg, args.precision, U, eta, args.sample_iters)
        cpu = {"value": gf, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": f"{its} CG iterations + final D-dagger of config {cfg.index} ({cfg.name}), fp64 oracle, full lattice"}
    del U, eta

    # ---------------- the other half of BASELINE.json's target statement: 32^4 in fp32 and fp64 (configs[3])
    also = []
    if not args.no_also and args.config == 4 and args.precision == 32:
        for prec in (32, 64):
            c3 = inputs.CONFIGS[3]
            a = time_device_resident(torch, wilson, c3, prec, max(args.steps, 5), max(args.warmup, 3), local, dist, world)
            k3, it3 = kernel_table(a["prof"], prec, a["V"], peak)
            also.append({"workload": workload_name(c3, a["r_min"]), "dtype": "f32" if prec == 32 else "f64",
                         "value": a["value"], "unit": "GFLOP/s", "ms_per_step": a["ms_step"], "steps": max(args.steps, 5),
                         "cg_iterations": a["iters"], "tile": a["tile"], "cg_iteration": it3, "kernels": k3,
                         "traffic_a3": stored_traffic(3, prec), "clocks": a["clocks"], "gpu_launches": a["launches"]})

    ws_bytes = (72 + 24 * 6) * V * (4 if args.precision == 32 else 8)
    line = {
        "metric": METRIC, "value": m["value"], "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": m["ms_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if args.precision == 32 else "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, r_min), "volume": V, "cg_iterations": m["iters"], "tile": m["tile"],
                   "l2_policy": f"inputs larger than L2 (working set {ws_bytes / 1e6:.0f} MB vs 126 MB L2)"
                   if ws_bytes > 2 * 126e6 else "working set fits L2 (latency-bound regime, no roofline claim)",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clocks": m["clocks"], "e2e": e2e, "gpu_launches": m["launches"], "roofline": roofline, "cpu_baseline": cpu,
        "also": also,
        "build": ({k: (len(v) if isinstance(v, list) else v) for k, v in wbuild.last_report().items() if k != "flags"}
                  if rank == 0 else None),
    }
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
