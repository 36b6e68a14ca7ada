"""bench.py prints ONE JSON line with the keys the driver reads (both arms)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
        "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches"}


def _run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_is_the_oracle_on_host_cores():
    r = _run("--impl", "reference", "--workload", "c2", "--steps", "2", "--warmup", "1", "--cpu-seconds", "1")
    assert BASE <= set(r) and r["impl"] == "reference" and r["gpu_launches"] == 0
    assert r["cpu_baseline"]["kind"] == "oracle" and r["cpu_baseline"]["cores"] >= 1 and r["cpu_baseline"]["value"] == r["value"] > 0
    assert r["e2e"] == {"value": r["value"], "unit": r["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert r["vs_baseline"] is None and r["unit"] == "GB/s" and r["higher_is_better"] is True


def test_reference_arm_other_ranks_stay_silent():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1"],
                         capture_output=True, text=True, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


@pytest.mark.gpu
def test_our_arm_line():
    r = _run("--steps", "5", "--warmup", "3", "--cpu-seconds", "2", "--e2e-steps", "1")
    assert BASE | {"roofline", "cpu_baseline", "clocks"} <= set(r)
    assert r["n_gpus"] == 1 and r["steps"] == 5 and r["gpu_launches"] == 15 and r["dtype"] == "u8" and r["data"] == "synthetic"
    assert r["config"]["workload"].startswith("c4") and "model" not in r["config"]
    ro = r["roofline"]
    assert ro["bound"] == "hbm" and ro["unit"] == "GB/s" and abs(ro["frac"] - ro["achieved"] / ro["peak"]) < 1e-9
    assert 0.7 * 8000 <= ro["achieved"] <= 8000 and 0.95 <= ro["traffic"] / ro["algorithmic_bytes"] <= 1.02
    assert r["e2e"]["h2d_bytes_per_step"] == r["e2e"]["d2h_bytes_per_step"] == 3 * 2 ** 29 and 0 < r["e2e"]["value"] < r["value"]
    assert r["cpu_baseline"]["kind"] == "oracle" and 0 < r["cpu_baseline"]["value"] < r["value"]
    assert not set(r["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}


@pytest.mark.gpu
def test_sharded_mode_degenerates_to_one_rank():
    """bench.py --mode sharded on one GPU: the multi-process executor with a world of 1 (every virtual device on rank 0)"""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0", MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--mode", "sharded", "--workload", "c2", "--steps", "5"],
                         capture_output=True, text=True, cwd=ROOT, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    r = json.loads([l for l in out.stdout.splitlines() if l.strip()][-1])
    assert r["mode"] == "sharded" and r["n_gpus"] == 1 and r["gpu_launches"] == 5 and r["scaling"] == "strong"
    assert r["rank0_bytes_per_step"] == 2 * 128 * 2 ** 20 and r["rank0_peer_destinations"] == 0 and r["value"] > 1000
