"""-m gpu: bench.py prints ONE JSON line that carries every key of the measurement contract, on a short run."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    return json.loads(lines[0])


def test_default_arm_line_has_the_contract_keys():
    d = run_bench("--steps", "20", "--warmup", "5", "--cpu-budget", "2", "--e2e-steps", "4", "--max-repeats", "9")
    assert d["metric"] == "env_steps_per_sec" and d["unit"] == "env-steps/s" and d["n_gpus"] == 1 and d["steps"] == 20 and d["warmup"] == 5
    assert d["higher_is_better"] is True and d["scaling"] == "weak" and d["vs_baseline"] is None and d["dtype"] == "f32" and d["data"] == "synthetic"
    assert "config 5" in d["config"]["workload"] and "65536" in d["config"]["workload"] and "l2" in d["config"]
    assert 0.010 < d["ms_per_step"] < 0.040 and d["repeats"] >= 7 and d["steps_per_timed_interval"] >= 100
    assert abs(d["value"] - 65536 / (d["ms_per_step"] * 1e-3)) / d["value"] < 1e-6
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and 0.3 < r["frac"] < 1.0
    assert r["traffic"] > 0 and r["traffic_timed"] > 0 and "x2" in r["kernel"] and 0.2 < r["hbm"]["frac"] < 1.0
    assert abs(r["flops_per_launch"] / (65536 * 4) - 3871.75) < 10.0            # the oracle's tally per drone and step (a few compares depend on the data)
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["single_thread_value"] > 0 and "envs" in c["sample"]
    e = d["e2e"]
    assert e["unit"] == "env-steps/s" and e["h2d_bytes_per_step"] == 65536 * 4 * 16 and e["d2h_bytes_per_step"] == 65536 * (64 * 4 + 5)
    assert 0 < e["value"] < d["value"]
    assert d["gpu_launches"] >= 20 * d["repeats"]
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons", "samples"}
    assert d["graph"]["ms_per_step"] > 0 and d["camera"]["roofline"]["bound"] == "hbm" and d["camera"]["rgba"]["us_per_call"] > 0


def test_reference_arm_line():
    d = run_bench("--impl", "reference", "--steps", "3", "--warmup", "1")
    assert d["impl"] == "reference" and d["metric"] == "env_steps_per_sec" and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "env-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
