"""Builds paper_2604_09184_b200/libnbkick.so in-tree with nvcc for sm_100a (no GPU needed)."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libnbkick.so")
SOURCES = [os.path.join(_CSRC, "nbkick.cu")]
HEADERS = [os.path.join(_CSRC, f) for f in ("nb_common.cuh", "force_tiles.cuh", "force_sym.cuh", "body_kernels.cuh", "kepler.cuh", "groups.cuh", "encounter.cuh", "merge.cuh", "sort_staging.cuh", "multilevel.cuh", "force_mixed.cuh", "force_symds.cuh", "step_small.cuh")] + [
    os.path.join(os.path.dirname(_HERE), "include", "nbkick.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
    "-Xptxas", "-v",
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        cmd = [nvcc(), *NVCC_FLAGS, "-o", LIB, *SOURCES]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed building libnbkick.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
