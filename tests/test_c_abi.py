"""The boundary is a C ABI: a plain-C program (tests/c_abi_smoke.c, gcc, no C++ and no torch) includes include/tt.h,
links libtt.so and runs the impulse-response check on the GPU."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = os.path.join(ROOT, "paper_2501_14911_b200")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def _build(tmp_path):
    from paper_2501_14911_b200 import build
    build.build()
    exe = str(tmp_path / "c_abi_smoke")
    cmd = ["gcc", "-std=c11", "-O1", os.path.join(ROOT, "tests", "c_abi_smoke.c"), "-I", os.path.join(ROOT, "include"),
           "-I", os.path.join(CUDA, "include"), "-L", PKG, "-ltt", "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-lm",
           "-Wl,-rpath," + PKG, "-Wl,-rpath," + os.path.join(CUDA, "lib64"), "-o", exe]
    subprocess.run(cmd, check=True, capture_output=True)
    return exe


@pytest.mark.skipif(shutil.which("gcc") is None, reason="needs gcc")
def test_header_compiles_as_c_and_links(tmp_path):
    """CPU-only: tt.h is valid C11 and every symbol the C program uses resolves against libtt.so."""
    _build(tmp_path)


@pytest.mark.gpu
def test_c_program_runs_the_path(tmp_path):
    exe = _build(tmp_path)
    res = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stdout + res.stderr
    assert "impulse response" in res.stdout
