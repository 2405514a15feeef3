"""-m gpu: the measurement contract of bench.py on a small workload (BASELINE config 1, 8^4, seconds): one JSON line on stdout
with the keys the driver parses, the device-resident value, the end-to-end value through host buffers, the per-kernel roofline
table and a positive count of this repo's kernel launches."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, cwd=ROOT,
                         timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines          # exactly ONE JSON line
    return json.loads(lines[0])


def test_bench_line_small_workload():
    d = _run("--config", "1", "--steps", "2", "--warmup", "3", "--sample-iters", "2")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "also"):
        assert k in d, k
    assert d["unit"] == "GFLOP/s" and d["higher_is_better"] is True and d["n_gpus"] == 1 and d["steps"] == 2
    assert d["dtype"] == "f32" and d["data"] == "synthetic" and d["vs_baseline"] is None and d["scaling"] == "weak"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["gpu_launches"] >= 2
    assert "workload" in d["config"] and "8^4" in d["config"]["workload"] and "model" not in d["config"]
    e = d["e2e"]
    assert e["value"] > 0 and e["value"] < 1.5 * d["value"] and e["steps"] == d["steps"]
    assert e["h2d_bytes_per_step"] == 4096 * (72 + 24) * 4 and e["d2h_bytes_per_step"] == 4096 * 24 * 4
    # value = the K steps pipelined over two contexts; the same steps as K cg_solve_host calls beside it
    assert "pipelined" in e["mode"] and e["outputs_identical"] is True
    assert e["one_call_at_a_time"]["value"] > 0 and e["one_call_at_a_time"]["ms_per_step"] > 0
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] > 1000
    assert len(r["kernels"]) == 3 and [k["name"][:2] for k in r["kernels"]] == ["a2", "a3", "a4"]
    assert r["kernels"][1]["bytes_per_launch"] == 576 * 4096
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and "sample" in c
    assert d["also"] == []                 # the 32^4 entries belong to the default workload only
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}


def test_bench_reference_arm_line():
    d = _run("--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "1")
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["gpu_launches"] == 0
