"""bench.py --impl reference (the CPU oracle arm) runs without a GPU and reports a consistent line."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _ref(*args):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", *args], capture_output=True,
                       text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    return json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1])


def test_reference_arm_full_evaluations_at_config0():
    line = _ref("--config", "0", "--steps", "2", "--warmup", "1")
    assert line["impl"] == "reference" and line["steps"] == 2 and line["warmup"] == 1 and line["gpu_launches"] == 0
    assert line["config"]["workload"] == "config0" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["value"] == line["value"] and line["e2e"]["h2d_bytes_per_step"] == 0
    # a step is a whole evaluation here: the real step time and the per-evaluation time agree
    assert abs(line["ms_per_step"] / 1e3 - line["seconds_per_eval_extrapolated"]) <= 0.05 * line["ms_per_step"] / 1e3 + 0.01


def test_reference_arm_bounded_sample_at_config2():
    """Configs 2-4 time a bounded sample (seconds) and extrapolate: ms_per_step is the sample's real time."""
    line = _ref("--config", "2", "--steps", "1", "--warmup", "0")
    assert line["ms_per_step"] < 120e3
    assert line["seconds_per_eval_extrapolated"] > 100 * line["ms_per_step"] / 1e3
    assert abs(line["value"] * line["seconds_per_eval_extrapolated"] - 1.0) < 1e-9
    assert "first 256 of 2000 outer ERI-grid points" in line["cpu_baseline"]["sample"]
