"""Build step: compile csrc/*.cu into paper_2302_01293_b200/libqlp_bls.so for sm_100a with nvcc.

The library is built in-tree so that it travels with the repository snapshot to the GPU box.
Usage: ``python -m paper_2302_01293_b200.build [--force]``.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libqlp_bls.so")
LIB_CHECK = os.path.join(_HERE, "libqlp_bls_check.so")   # the same sources with -DQLP_BOUNDS_CHECK (tests only)
UBENCH = os.path.join(_HERE, "qlp_ubench")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
                  [os.path.join(os.path.dirname(_HERE), "include", "qlp_bls.h")])


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def build_check(force: bool = False) -> str:
    """The bounds-check build (include/qlp_bls.h qlp_bls_debug_violations): same sources, -DQLP_BOUNDS_CHECK."""
    t = os.path.getmtime(LIB_CHECK) if os.path.exists(LIB_CHECK) else 0.0
    if force or any(os.path.getmtime(s) > t for s in sources()):
        nvcc = os.environ.get("NVCC", "nvcc")
        subprocess.run([nvcc, *NVCC_FLAGS, "-DQLP_BOUNDS_CHECK", "-o", LIB_CHECK, os.path.join(CSRC, "api.cu")],
                       check=True)
    return LIB_CHECK


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc, *NVCC_FLAGS, "-o", LIB, os.path.join(CSRC, "api.cu")]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.run(cmd, check=True)
    src = os.path.join(CSRC, "ubench.cu")
    if force or not os.path.exists(UBENCH) or os.path.getmtime(UBENCH) < os.path.getmtime(src):
        nvcc = os.environ.get("NVCC", "nvcc")
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                        "-cudart", "static", "-o", UBENCH, src], check=True)
    return LIB


if __name__ == "__main__":
    if "--check" in sys.argv:
        print(build_check(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
