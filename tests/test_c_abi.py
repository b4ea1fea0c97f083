"""include/vs.h as a C99 header: tests/c_abi_smoke.c is compiled with gcc -std=c99 (no C++, no Python in between), linked
against libvs_b200.so and -- on a GPU box -- run."""
import os
import subprocess
import sys

import pytest

from paper_2409_02482_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def _build(tmp_path):
    binding.load_library()          # builds libvs_b200.so if it is stale
    exe = str(tmp_path / "c_abi_smoke")
    libdir = os.path.dirname(binding.LIB_PATH)
    cmd = ["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", "-I", os.path.join(ROOT, "include"),
           "-isystem", os.path.join(CUDA, "include"), os.path.join(ROOT, "tests", "c_abi_smoke.c"), "-o", exe,
           "-L", libdir, "-l:libvs_b200.so", "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-lm",
           "-Wl,-rpath," + libdir, "-Wl,-rpath," + os.path.join(CUDA, "lib64")]
    res = subprocess.run(cmd, capture_output=True, text=True)
    assert res.returncode == 0, res.stdout + res.stderr
    return exe


def test_header_is_c99_and_links(tmp_path):
    """CPU-only part: the header compiles as strict C99 and every symbol the C caller uses resolves at link time."""
    _build(tmp_path)


@pytest.mark.gpu
def test_c_caller_renders_the_closed_form_quad(tmp_path):
    exe = _build(tmp_path)
    res = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    sys.stdout.write(res.stdout)
    assert res.returncode == 0, res.stdout + res.stderr
    assert "c_abi_smoke ok" in res.stdout
