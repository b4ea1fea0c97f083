"""Compile oracle/vs_oracle.c into oracle/libvs_oracle.so with gcc (TEST INFRASTRUCTURE).

Flags: no FMA contraction, no fast-math, so the fp32-exact steps are IEEE.
`python -m oracle.build` or `oracle.build.ensure_built()`.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "vs_oracle.c")
LIB = os.path.join(HERE, "libvs_oracle.so")
FLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
         "-Wall", "-Wextra", "-Wno-unused-parameter"]


def ensure_built(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        tmp = LIB + ".tmp%d" % os.getpid()
        subprocess.run(["gcc", *FLAGS, SRC, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(ensure_built(force=True))
