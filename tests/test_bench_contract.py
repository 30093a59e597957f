"""The bench.py line of the reference (oracle) arm carries the keys the measurement contract names.
The CUDA arm needs a GPU and is exercised by the driver; its keys are checked in the gpu-marked test."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
        "vs_baseline", "dtype", "data", "config", "e2e"}


def _line(args, timeout):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True,
                         timeout=timeout, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1, "bench.py must print exactly one line"
    return json.loads(lines[0])


def test_reference_arm_line():
    d = _line(["--impl", "reference", "--steps", "1", "--warmup", "0", "--cpu-seconds", "1"], 300)
    assert BASE <= set(d) and d["impl"] == "reference"
    assert d["metric"].startswith("geodesics/sec") and d["unit"] == "geodesics/s" and d["dtype"] == "f64"
    assert d["config"]["workload"] == "headline" and d["higher_is_better"] is True and d["vs_baseline"] is None
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and "rays of headline" in cb["sample"] and cb["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "geodesics/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["value"] > 1e3


@pytest.mark.gpu
def test_cuda_arm_line():
    d = _line(["--steps", "3", "--warmup", "3", "--cpu-seconds", "2"], 600)
    assert BASE | {"roofline", "cpu_baseline", "clocks", "gpu_launches", "tail"} <= set(d)
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert d["gpu_launches"] == 3 and d["n_gpus"] == 1 and d["scaling"] == "weak"
    # both flop models, best and median, the counter evidence with its source
    assert "SURVEY.md 8(d): 70/RHS + 330/step" in r["flop_model"] and r["frac_builder_model"] > r["frac"]
    assert r["profile"] and os.path.exists(os.path.join(ROOT, r["profile"])) and r["traffic"] and 0.3 < r["hw_fp64_frac"] < 1.0
    assert d["ms_per_step_best"] <= d["ms_per_step_median"] <= 1.5 * d["ms_per_step"]
    assert d["back_to_back"]["images"] == 8 and d["back_to_back"]["ms_per_image"] < 1.05 * d["ms_per_step"]
    assert d["cpu_baseline"]["single_thread"]["value"] < d["cpu_baseline"]["value"]
    assert d["config"]["workload"] == "headline" and d["dtype"] == "f64"
    assert d["e2e"]["d2h_bytes_per_step"] >= 1024 * 1024 * 128 and d["e2e"]["value"] > 0.5 * d["value"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 100 * d["cpu_baseline"]["value"]
    assert d["clocks"]["sm_mhz"] > 0 and not set(d["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown",
                                                                           "sw_thermal_slowdown"}
