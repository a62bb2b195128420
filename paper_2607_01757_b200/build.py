"""Builds libdkd.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libdkd.so")
SOURCES = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith(".cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cuh", ".h"))] + [
    os.path.join(ROOT, "include", "dkd.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC", "-cudart", "static",
]


def nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


LIB_DEBUG = os.path.join(_HERE, "libdkd_debug.so")


def build(force: bool = False, verbose: bool = False, debug: bool = False) -> str:
    """Builds libdkd.so, or with debug=True libdkd_debug.so: the same sources with -DDKD_DEBUG, i.e. device-side
    bounds checks (assert) on every workspace / shared-memory index and on the mbarrier ring arithmetic.  The GPU
    tests run their random sweep and worst-case inputs under it (DKD_LIBRARY=libdkd_debug.so)."""
    lib = LIB_DEBUG if debug else LIB
    stale = force or not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in DEPS)
    if stale:
        tmp = lib + f".tmp{os.getpid()}"
        cmd = [nvcc(), *NVCC_FLAGS, "-I", os.path.join(ROOT, "include"), "-I", CSRC]
        if debug:
            cmd += ["-DDKD_DEBUG"]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += [*SOURCES, "-o", tmp]
        subprocess.check_call(cmd)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, debug="--debug" in sys.argv))
