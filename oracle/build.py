"""Compile oracle/vs_oracle.c into oracle/libvs_oracle.so with gcc (TEST INFRASTRUCTURE).

Flags: no FMA contraction, no fast-math, so the fp32-exact steps are IEEE.
`python -m oracle.build` or `oracle.build.ensure_built()`.

With VS_ORACLE_SANITIZE=1 in the environment the oracle is built with AddressSanitizer + UndefinedBehaviorSanitizer into a
file of its own and that build is the one loaded; the interpreter is not instrumented, so run it as
    VS_ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
        python -m pytest tests -q -m "not gpu" -k oracle
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "vs_oracle.c")
LIB = os.path.join(HERE, "libvs_oracle.so")
FLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
         "-Wall", "-Wextra", "-Wno-unused-parameter"]


SAN_LIB = os.path.join(HERE, "libvs_oracle_san.so")
SAN_FLAGS = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]


def ensure_built(force: bool = False) -> str:
    sanitize = os.environ.get("VS_ORACLE_SANITIZE", "") not in ("", "0")
    lib = SAN_LIB if sanitize else LIB
    flags = [f for f in FLAGS if f != "-O2"] + SAN_FLAGS if sanitize else FLAGS
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(SRC):
        tmp = lib + ".tmp%d" % os.getpid()
        subprocess.run(["gcc", *flags, SRC, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(ensure_built(force=True))
