"""bench.py on the GPU box: one JSON line with every key of the measurement contract (pytest -m gpu)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*extra):
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *extra], capture_output=True, text=True,
                         timeout=900, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def test_default_workload_line():
    d = run_bench("--steps", "60", "--warmup", "3")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in d, k
    assert d["config"]["workload"] == "config4_bandwidth_stress" and d["dtype"] == "f64" and d["n_gpus"] == 1
    assert d["steps"] == 60 and d["gpu_launches"] == 20                       # 3 time steps per launch
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert r["kernel"] == "sweep_kernel" and r["traffic"] and 0.3 < r["frac"] < 1.1
    assert r["one_step_per_pass"]["launches"] == r["one_step_per_pass"]["steps"]
    assert 0.5 < r["one_step_per_pass"]["frac"] < 1.1                         # the HBM-bound form of the kernel
    e = d["e2e"]
    assert e["unit"] == d["unit"] and 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] > 0 < e["d2h_bytes_per_step"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and 0 < cb["value"] < d["value"]
    assert d["clocks"] is None or set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert abs(d["check"]["norm"] - 1.0) < 1e-10


def test_resident_workload_line():
    d = run_bench("--workload", "1", "--steps", "400", "--warmup", "3", "--no-cpu-baseline")
    assert d["gpu_launches"] == 1 and d["roofline"]["kernel"] == "resident_kernel" and d["roofline"]["bound"] == "alu"
    assert d["e2e"]["value"] > 0 and abs(d["check"]["norm"] - 1.0) < 1e-10
