"""The boundary is C: include/reshard.h must compile as C99, and a program written in plain C against it must
link with libreshard.so and run (host-only here; with the kernels on the GPU box)."""
import os
import subprocess

import pytest

from paper_2211_05322_b200 import reshard as rs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "c_abi", "abi_smoke.c")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def _build(tmp_path):
    exe = str(tmp_path / "abi_smoke")
    libdir = os.path.dirname(rs.LIB_PATH)
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                    "-isystem", os.path.join(CUDA, "include"), SRC, "-o", exe, "-L", libdir, "-l:libreshard.so",
                    "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-Wl,-rpath," + libdir,
                    "-Wl,-rpath," + os.path.join(CUDA, "lib64")], check=True)
    return exe


def test_header_is_c99_and_host_calls_work_from_c(tmp_path):
    rs._lib()                                                  # make sure the library is built
    out = subprocess.run([_build(tmp_path)], capture_output=True, text=True)
    assert out.returncode == 0, out.stderr
    assert "c abi ok (host only" in out.stdout


@pytest.mark.gpu
def test_c_program_runs_the_kernels(tmp_path):
    out = subprocess.run([_build(tmp_path), "gpu"], capture_output=True, text=True)
    assert out.returncode == 0, out.stderr
    assert "c abi ok (gpu" in out.stdout
