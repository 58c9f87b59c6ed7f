"""Builds libmc_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libmc_b200.so")
SOURCES = [os.path.join(CSRC, "mc_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "mc_kernels.cuh"), os.path.join(CSRC, "mc_device.cuh"), os.path.join(CSRC, "mc_tile.cuh"),
                  os.path.join(os.path.dirname(_HERE), "include", "mc.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-ftz=true", "-prec-div=false", "-prec-sqrt=false",
    "-shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-O2",
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    tmp = f"{LIB}.{os.getpid()}.tmp"
    extra = os.environ.get("MC_B200_NVCC_EXTRA", "").split()      # experiments only (e.g. -DMC_TILE_MIN_BLOCKS=3)
    cmd = [nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
