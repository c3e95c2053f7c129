"""Build step: compiles the CUDA sources into paper_1208_0961_b200/libcuba.so for sm_100a.

    python -m paper_1208_0961_b200.build [--force]

-fmad=false is part of the arithmetic contract (A2): no fused multiply-add is
formed from separate fp64 operations, so the kernels round exactly where the paper-derived
operation order says.  -lineinfo keeps the ncu source page usable.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcuba.so")

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-fmad=false", "-Xcompiler", "-fPIC,-ffp-contract=off,-O2", "-shared",
    "-Xptxas", "-v",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def deps():
    return sources() + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [os.path.join(ROOT, "include", "cuba.h")]


# Test build: every element / pair / particle takes the rare exact paths (in-bucket ranking with
# pid tie-break, oracle-order Eq. 3 decision, exact direction of the fused histogram).  The GPU
# tests run the parity cases against it as well, so the fallbacks are covered bit for bit.
LIB_SLOW = os.path.join(HERE, "libcuba_slowpaths.so")


def _compile(lib: str, extra, force: bool, verbose: bool, log_name: str) -> str:
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps()):
        return lib
    tmp = lib + ".tmp.%d" % os.getpid()
    cmd = ["nvcc", *NVCC_FLAGS, *extra, "-o", tmp, *sources()]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(HERE, log_name), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if res.returncode != 0:
        sys.stderr.write(log)
        raise RuntimeError("nvcc failed")
    os.replace(tmp, lib)
    if verbose:
        print(log)
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    return _compile(LIB, [], force, verbose, "build.log")


def build_slowpaths(force: bool = False, verbose: bool = False) -> str:
    return _compile(LIB_SLOW, ["-DCUBA_FORCE_SLOW_PATHS=1"], force, verbose, "build_slowpaths.log")


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    print(build_slowpaths(force="--force" in sys.argv))
