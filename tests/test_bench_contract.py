"""bench.py prints ONE JSON line with the contract's keys: reference arm on CPU, our arm on the GPU."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "cpu_baseline"}


def _run(args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True, cwd=ROOT,
                       timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_line():
    d = _run(["--impl", "reference", "--workload", "config1", "--steps", "3", "--warmup", "1"])
    assert BASE_KEYS <= set(d)
    assert d["impl"] == "reference" and d["unit"] == "MLUPS" and d["dtype"] == "f64" and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"] == "config1" and d["value"] > 0 and d["gpu_launches"] == 0


def test_reference_arm_other_ranks_print_nothing():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "config1",
                        "--steps", "1", "--warmup", "0", "--gpus", "2"], capture_output=True, text=True, cwd=ROOT, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


@pytest.mark.gpu
def test_our_arm_line():
    d = _run(["--workload", "config5_128", "--steps", "6", "--warmup", "3"])
    assert BASE_KEYS | {"clocks", "roofline"} <= set(d)
    assert d["unit"] == "MLUPS" and d["dtype"] == "f64" and d["scaling"] == "weak" and d["higher_is_better"] is True
    assert d["gpu_launches"] == 12 and d["n_gpus"] == 1 and d["config"]["workload"] == "config5_128"
    rf = d["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s" and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    assert 0.2 < rf["frac"] < 1.2 and rf["ms_per_launch"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0 and 0 < d["e2e"]["value"] <= d["value"] * 1.05
    assert d["e2e"]["per_step_io"]["value"] < d["e2e"]["value"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}


@pytest.mark.gpu
def test_slab_overhead_line():
    d = _run(["--workload", "config5_128", "--slabs", "2", "--steps", "4", "--warmup", "3"])
    assert d["config"]["slabs"] == 2 and d["config"]["finite"] and d["value"] > 0
