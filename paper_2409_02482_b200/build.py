"""Build paper_2409_02482_b200/libvs_b200.so (the C-ABI library of include/vs.h) with nvcc for sm_100a.

`python -m paper_2409_02482_b200.build [--force] [--lib PATH] [-DNAME=VALUE ...]`.  `--lib` with -D switches builds a
variant of the same sources (the experiment switches of the kernels, e.g. -DVS_SHADE_PREFETCH=0) into another file, which
`bench.py --lib PATH` loads.  The .so is built IN-TREE so that it travels to the
GPU box with the repository snapshot; nvcc cross-compiles without a GPU.  Every .cu is compiled to an
object of its own (in parallel, cached under build/ by a hash of the source, the headers and the flags)
and the objects are linked into the shared library.
"""
from __future__ import annotations

import concurrent.futures
import glob
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvs_b200.so")
OBJ_DIR = os.path.join(HERE, "..", "build", "vs_b200")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [os.path.join(HERE, "..", "include", "vs.h")]


def _stale(lib: str) -> bool:
    if not os.path.exists(lib):
        return True
    return any(os.path.getmtime(d) > os.path.getmtime(lib) for d in sources() + _headers())


def _compile_one(nvcc, src, flags, header_digest, force):
    h = hashlib.sha256(header_digest)
    h.update(open(src, "rb").read())
    h.update(" ".join(flags).encode())
    obj = os.path.join(OBJ_DIR, "%s.%s.o" % (os.path.splitext(os.path.basename(src))[0], h.hexdigest()[:16]))
    log = obj + ".log"
    if force or not os.path.exists(obj) or not os.path.exists(log):
        tmp = obj + ".tmp%d" % os.getpid()
        res = subprocess.run([nvcc, *flags, "-c", src, "-o", tmp], capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s%s" % (src, res.stdout, res.stderr))
        os.replace(tmp, obj)
        open(log, "w").write(res.stderr)
    return obj, open(log).read()


def build(lib: str = LIB, extra_flags=(), force: bool = False, verbose: bool = False) -> str:
    """Compile and link `lib`.  `extra_flags` (e.g. -D switches of an experiment) are part of the object cache key."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ_DIR, exist_ok=True)
    flags = [*NVCC_FLAGS, *extra_flags]
    hd = hashlib.sha256()
    for hpath in _headers():
        hd.update(open(hpath, "rb").read())
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        results = list(ex.map(lambda s: _compile_one(nvcc, s, flags, hd.digest(), force), sources()))
    tmp = lib + ".tmp%d" % os.getpid()
    res = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", *[o for o, _ in results], "-o", tmp],
                         capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + res.stdout + res.stderr)
    os.replace(tmp, lib)
    if verbose:
        print("".join(log for _, log in results))
    return lib


def ensure_built(force: bool = False, verbose: bool = False) -> str:
    if force or _stale(LIB):
        build(LIB, force=force, verbose=verbose)
    return LIB


if __name__ == "__main__":
    argv = sys.argv[1:]
    if "--lib" in argv:
        out = os.path.abspath(argv[argv.index("--lib") + 1])
        defines = [a for a in argv if a.startswith("-D")]
        print(build(out, extra_flags=defines, force="--force" in argv, verbose=True))
    else:
        print(ensure_built(force="--force" in argv, verbose=True))
