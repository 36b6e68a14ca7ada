"""AddressSanitizer + UndefinedBehaviorSanitizer over everything that runs on the host (S5 "Sanitizers"):
the library's planner / scheduler / table builder / tile decode / pipeline simulator (the four host .cpp files, no
CUDA) and the C oracle, each driven by a small committed main under tests/sanitize/.  compute-sanitizer is closed on
the GPU pool, so the device side relies on the parity tests' guard bands instead."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2211_05322_b200", "csrc")
SAN = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]


def _run(exe):
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    out = r.stdout + r.stderr
    assert r.returncode == 0 and "runtime error" not in out and "AddressSanitizer" not in out and "LeakSanitizer" not in out, out[-4000:]
    return out


@pytest.mark.skipif(shutil.which("g++") is None, reason="needs g++")
def test_host_planner_under_asan_ubsan(tmp_path):
    exe = str(tmp_path / "host_planner_san")
    srcs = [os.path.join(CSRC, f) for f in ("plan.cpp", "schedule.cpp", "pipeline.cpp", "tables.cpp")]
    subprocess.run(["g++", "-std=c++17", "-Wall", "-Wextra"] + SAN + [os.path.join(ROOT, "tests", "sanitize", "host_planner_main.cpp")] + srcs +
                   ["-o", exe], check=True)
    out = _run(exe)
    assert " 0 failures" in out


@pytest.mark.skipif(shutil.which("gcc") is None, reason="needs gcc")
def test_oracle_under_asan_ubsan(tmp_path):
    exe = str(tmp_path / "oracle_san")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-fopenmp"] + SAN + [os.path.join(ROOT, "tests", "sanitize", "oracle_main.c"), "-o", exe],
                   check=True)
    out = _run(exe)
    assert " 0 failures" in out
