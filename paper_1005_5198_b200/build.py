"""Builds libmicrolens_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1005_5198_b200.build [--force]
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libmicrolens_b200.so")
SOURCES = [os.path.join(CSRC, "microlens.cu"), os.path.join(CSRC, "mapstats.cu")]
DEPENDS = SOURCES + [os.path.join(CSRC, "shoot_kernel.cuh"), os.path.join(_ROOT, "include", "microlens.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(s) > t for s in DEPENDS)


def build_library(force: bool = False, verbose: bool = False, defines=(), out: str = None) -> str:
    """Compile csrc/*.cu into libmicrolens_b200.so next to this file; returns its path.

    `defines` (e.g. ["ML_MAX_GRID_Y=50"]) and `out` make a separate TEST build of the same sources (the
    launch-split test uses one); such a build is loaded by pointing MICROLENS_B200_LIBRARY at it (binding.load)."""
    if defines and (out is None or os.path.abspath(out) == os.path.abspath(LIB_PATH)):
        # such a library would be newer than its sources, so is_stale() would keep it: every later load (bench, tests)
        # would silently run the test build
        raise ValueError("build_library: `defines` make a test build and need an `out` other than the shipped %s" % LIB_PATH)
    target = out or LIB_PATH
    if not out and not defines and not force and not is_stale():
        return LIB_PATH
    tmp = target + ".tmp%d" % os.getpid()
    cmd = ([_nvcc()] + NVCC_FLAGS + ["-D" + d for d in defines] + (["-Xptxas", "-v"] if verbose else [])
           + ["-o", tmp] + SOURCES)
    try:
        subprocess.check_call(cmd, cwd=_HERE)
        os.replace(tmp, target)
    finally:
        if os.path.exists(tmp):
            os.remove(tmp)
    return target


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
