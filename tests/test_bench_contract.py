"""bench.py prints ONE JSON line with the keys the driver reads (reference arm here on CPU, our arm on the GPU)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
COMMON = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
          "dtype", "data", "config", "e2e", "gpu_launches")


def _run(args, timeout):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=timeout, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout
    return json.loads(lines[0])


def test_reference_arm_line():
    d = _run(["--impl", "reference", "--steps", "1", "--warmup", "0"], 600)
    for k in COMMON + ("impl", "cpu_baseline"):
        assert k in d, k
    assert d["impl"] == "reference" and d["metric"] == "ssfm_grid_point_z_steps_per_s" and d["unit"] == "grid-point z-steps/s"
    assert d["value"] > 0 and d["higher_is_better"] is True and d["vs_baseline"] is None and d["dtype"] == "f64"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert "workload" in d["config"] and "model" not in d["config"]


@pytest.mark.gpu
def test_our_arm_line():
    d = _run(["--steps", "2", "--warmup", "3", "--rt-per-step", "2", "--no-cpu-baseline"], 600)
    for k in COMMON + ("clocks", "roofline", "round_trips_per_s"):
        assert k in d, k
    assert d["value"] > 1e9 and d["n_gpus"] == 1 and d["dtype"] == "f32" and d["scaling"] == "weak" and d["data"] == "synthetic"
    assert d["config"]["engine"] == "solo" and "C4" in d["config"]["workload"]      # what AUTO picks for a batch >= SM count
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and 0.05 < r["frac"] < 1.0
    assert d["gpu_launches"] == d["steps"]                      # one launch of the on-chip kernel per step
    assert d["e2e"]["h2d_bytes_per_step"] == 256 * 16384 * 8 * 3 and d["e2e"]["d2h_bytes_per_step"] == 256 * 16384 * 8
    assert d["e2e"]["value"] > 0 and d["e2e"]["value"] != d["value"]
    assert d["clocks"]["sm_mhz"] is None or d["clocks"]["sm_mhz"] > 0
