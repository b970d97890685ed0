"""bench.py prints ONE JSON line with the keys the driver reads (base contract + this tier's roofline / cpu_baseline)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches"}


def _run(args, timeout):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True,
                       timeout=timeout, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_line():
    """--impl reference: the oracle on the host cores, same metric / unit / config keys, rank 0 only."""
    d = _run(["--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0"], 300)
    assert BASE_KEYS <= set(d) and d["impl"] == "reference"
    assert d["metric"] == "near_field_pair_interactions_per_s" and d["unit"] == "interactions/s"
    assert d["config"]["workload"] == "config1_uniform_32" and d["dtype"] == "f64" and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["value"] > 0 and d["higher_is_better"] is True and d["vs_baseline"] is None


@pytest.mark.gpu
def test_b200_arm_line():
    d = _run(["--config", "1", "--steps", "3", "--warmup", "3", "--per-config", "", "--no-cpu-baseline"], 600)
    assert BASE_KEYS | {"clocks", "roofline", "particle_updates_per_s"} <= set(d)
    assert d["config"]["workload"] == "config1_uniform_32" and d["dtype"] == "f32" and d["data"] == "synthetic"
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["scaling"] == "weak"
    rf = d["roofline"]
    assert rf["bound"] == "alu" and rf["unit"] == "TFLOP/s" and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert abs(rf["peak"] - rf["sm_count"] * 128 * 2 * rf["clock_khz"] * 1e3 / 1e12) < 1e-9
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 12 * d["config"]["n"] == e["d2h_bytes_per_step"] and 0 < e["value"] <= d["value"] * 1.05
    assert d["gpu_launches"] >= 3 * 2 and {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])
    assert d["sum_check"] < 1e-6
    assert d["fused_density"]["mean_rho"] >= 1.0 and d["fused_kick"]["max_accel"] > 0
