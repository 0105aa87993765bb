"""bench.py prints ONE JSON line with the keys of the measurement contract (metric/value/unit, roofline, e2e, cpu_baseline,
gpu_launches, clocks), and the reference arm prints its own line.  Runs the real script on the GPU with few steps."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(*extra):
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *extra], capture_output=True, text=True, cwd=ROOT,
                         timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_bench_line_contract():
    d = run("--steps", "4", "--warmup", "3")
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert key in d, key
    assert d["n_gpus"] == 1 and d["steps"] == 4 and d["warmup"] == 3 and d["dtype"] == "bf16" and d["vs_baseline"] is None
    assert "workload" in d["config"] and "configs[2]" in d["config"]["workload"]
    r = d["roofline"]
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-3
    assert r["traffic"] is None or r["traffic"] > 0
    assert 0.3 < r["frac"] < 1.0 and d["value"] > 500
    assert d["gpu_launches"] == 4                                   # one fused launch per timed step
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] > 3e8 and e["d2h_bytes_per_step"] > 1e8 and 0 < e["value"] < d["value"]
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"]
    for leg in ("append", "migrate"):
        assert d[leg]["bound"] == "hbm" and 0.3 < d[leg]["frac"] <= 1.05
    for leg in ("d2h", "h2d"):
        assert 0.5 < d["offload"][leg]["frac"] <= 1.05 and 0.5 < d["offload"]["scattered"][leg]["frac"] <= 1.05
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}


def test_reference_arm_line():
    d = run("--impl", "reference", "--steps", "1", "--warmup", "1")
    assert d["impl"] == "reference" and d["dtype"] == "f64" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
