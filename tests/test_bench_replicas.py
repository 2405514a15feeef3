"""Host logic of bench.py for N > 1 (-m "not gpu"): the path does not shard ("replicas only"), so
the multi-GPU number is N independent solves, timed as the max over ranks.  Covered here with world_size 2 on
the gloo backend: the max-over-ranks reduction, the whole-job aggregate, and that under a 2-rank launch only
rank 0 of the reference arm prints a line."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 100.0 + 25.0 * rank                      # rank 1 is the slow one
    got = bench.max_over_ranks(ms, dist, "cpu")
    val = bench.whole_job_value(world, 4096, 83, got * 1e-3)
    dist.barrier()
    out[rank] = (got, val)
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_world_size_2():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    assert out[0] == out[1]
    t, v = out[0]
    assert t == 125.0
    one = bench.cg_flops(4096, 83) / 0.125 / 1e9
    assert abs(v - 2 * one) < 1e-9 * v


def test_single_rank_paths_need_no_process_group():
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.cg_flops(256, 28) == 256 * (2976 * 28 + 1368)


def test_reference_arm_prints_on_rank_0_only():
    env = dict(os.environ, WORLD_SIZE="2", OMP_NUM_THREADS="2")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
           "--steps", "1", "--warmup", "0", "--gpus", "2"]
    r1 = subprocess.run(cmd, env=dict(env, RANK="1"), capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(env, RANK="0"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["unit"] == "GFLOP/s" and line["higher_is_better"] is True
