"""k_raster_direct divides by the triangle's area with the reciprocal hoisted out of its per-sample loop (csrc/vs_div.cuh).
DESIGN.md 3.4 wants the IEEE quotient (the oracle divides in C): tests/fdiv_check.cu compares the seeded sequence with
__fdiv_rn, bit for bit, on every divisor a small triangle can have."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def _build(tmp_path):
    exe = str(tmp_path / "fdiv_check")
    res = subprocess.run([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", os.path.join(ROOT, "tests", "fdiv_check.cu"), "-o", exe],
                         capture_output=True, text=True)
    assert res.returncode == 0, res.stdout + res.stderr
    return exe


def test_fdiv_check_compiles(tmp_path):
    _build(tmp_path)


@pytest.mark.gpu
def test_seeded_division_is_the_ieee_division(tmp_path):
    exe = _build(tmp_path)
    res = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    sys.stdout.write(res.stdout)
    assert res.returncode == 0, res.stdout + res.stderr
    assert "fdiv_check ok" in res.stdout
