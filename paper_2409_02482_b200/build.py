"""Build paper_2409_02482_b200/libvs_b200.so (the C-ABI library of include/vs.h) with nvcc for sm_100a.

`python -m paper_2409_02482_b200.build [--force]`.  The .so is built IN-TREE so that it travels to the
GPU box with the repository snapshot; nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvs_b200.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "vs.h")]
    return any(os.path.getmtime(d) > os.path.getmtime(LIB) for d in deps)


def ensure_built(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + ".tmp%d" % os.getpid()
        cmd = [nvcc, *NVCC_FLAGS, *sources(), "-o", tmp]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
        os.replace(tmp, LIB)
        if verbose:
            print(res.stderr)
    return LIB


if __name__ == "__main__":
    print(ensure_built(force="--force" in sys.argv, verbose=True))
