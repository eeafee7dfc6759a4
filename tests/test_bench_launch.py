"""bench.py launch plumbing: `--gpus N` must create N ranks (or fail loudly), never run silently on one GPU."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu


def _bench(*args, timeout=900):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE")}
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                          timeout=timeout, env=env, cwd=ROOT)


def test_gpus_2_spawns_two_ranks_or_fails_loudly():
    import torch
    r = _bench("--gpus", "2", "--config", "1", "--steps", "2", "--warmup", "3", "--no-cpu-baseline")
    if torch.cuda.device_count() < 2:
        assert r.returncode != 0 and "--gpus 2 requested" in (r.stdout + r.stderr)
        return
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "strong" and line["value"] > 0


def test_bench_line_small_config():
    r = _bench("--config", "0", "--steps", "3", "--warmup", "3")
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1])
    for key in ("metric", "value", "e2e", "roofline", "rooflines_by_class", "cpu_baseline", "clocks", "gpu_launches", "extra"):
        assert key in line, key
    assert line["config"]["workload"] == "config0" and line["gpu_launches"] > 0 and line["e2e"]["value"] > 0
    assert set(line["extra"]["yardstick"]) >= {"thc_dgemm_8192_tflops", "torch_matmul_fp64_8192_tflops"}
