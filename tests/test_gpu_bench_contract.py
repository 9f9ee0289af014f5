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
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks",
              "configs"):
        assert k in d, k
    assert d["config"]["workload"] == "config4_bandwidth_stress" and d["dtype"] == "f64" and d["n_gpus"] == 1
    assert set(d["config"]) == {"workload", "n_harm", "n_phiy", "n_batch", "dt", "name", "n_steps", "note"}   # = reference arm's
    r = d["roofline"]
    S = round(r["steps_per_launch"])
    assert d["steps"] == 60 and d["gpu_launches"] == 60 // S and S in (2, 3, 4)     # S time steps per launch
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert r["kernel"] in ("sweep_kernel", "warpsweep_kernel") and 0.3 < r["frac"] < 1.1
    assert r["one_step_per_pass"]["launches"] == r["one_step_per_pass"]["steps"]
    f32 = d["other_precisions"]["f32_storage"]        # NEXT-4 leg beside the headline: same kernel, fp32 pairs in HBM
    assert f32["dtype"] == "f32 storage / f64 arithmetic" and f32["kernel"] == "warpsweep_kernel" and f32["value"] > 0
    assert abs(f32["check"]["norm"] - 1.0) < 1e-4 and f32["steps"] == 60
    assert 0.5 < r["one_step_per_pass"]["frac"] < 1.1                         # the HBM-bound form of the kernel
    e = d["e2e"]
    assert e["unit"] == d["unit"] and 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] > 0 < e["d2h_bytes_per_step"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and 0 < cb["value"] < d["value"]
    # the clock record must exist on the GPU box: median SM clock under load, max clock, throttle reasons
    c = d["clocks"]
    assert c is not None and c["samples"] >= 5 and c["sm_mhz"] > 0 and c["sm_max_mhz"] >= c["sm_mhz"] and isinstance(c["reasons"], list)
    assert abs(d["check"]["norm"] - 1.0) < 1e-10
    # every other BASELINE config is timed in the same run, with its own norm check
    assert set(d["configs"]) == {"config3_batched_sweep", "config2_paper_scale", "config1_crossed_ac", "config0_dc_B0"}
    for name, c in d["configs"].items():
        assert c["value"] > 0 and c["gpu_launches"] >= 1 and abs(c["check"]["norm"] - 1.0) < 1e-9, name
        assert c["roofline"]["bound"] in ("hbm", "alu") and 0 < c["roofline"]["frac"] < 1.2, name
    assert d["configs"]["config3_batched_sweep"]["roofline"]["bound"] == "hbm"
    assert d["configs"]["config0_dc_B0"]["roofline"]["kernel"] == "resident_kernel"


def test_resident_workload_line():
    d = run_bench("--workload", "1", "--steps", "400", "--warmup", "3", "--no-cpu-baseline", "--no-other-configs")
    assert d["gpu_launches"] == 1 and d["roofline"]["kernel"] == "resident_kernel" and d["roofline"]["bound"] == "alu"
    assert d["e2e"]["value"] > 0 and abs(d["check"]["norm"] - 1.0) < 1e-10


def test_cross_check_variant_is_labelled_by_what_ran():
    d = run_bench("--steps", "6", "--warmup", "3", "--variant", "1", "--no-cpu-baseline", "--no-other-configs")
    r = d["roofline"]
    assert r["kernel"].startswith("half_update_kernel") and d["gpu_launches"] == 18     # 3 launches per step
    assert abs(r["algorithmic_bytes_per_launch"] - 96.0 * 513 * 32001) < 1.0          # 96 B per point and step
