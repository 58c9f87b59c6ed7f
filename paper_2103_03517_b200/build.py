"""Builds libmc_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

One object per translation unit (compiled in parallel), then one link: the kernels of the generic pass, the pair pass and
the staged passes each live in their own .cu so that a change to one does not rebuild the others.
"""
from __future__ import annotations

import glob
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJDIR = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "libmc_b200.so")
HEADERS = sorted(glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h"))) + [os.path.join(os.path.dirname(_HERE), "include", "mc.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-ftz=true", "-prec-div=false", "-prec-sqrt=false",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-O2",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False, extra=(), lib: str = LIB, objdir: str = OBJDIR) -> str:
    """Compiles what is out of date and links ``lib``.  ``extra`` (additional nvcc flags, e.g. ``-DMC_X=1``) and a different
    ``lib`` / ``objdir`` are for experiment builds next to the product library; the product build passes none."""
    os.makedirs(objdir, exist_ok=True)
    tag = hashlib.sha1(" ".join(list(NVCC_FLAGS) + list(extra)).encode()).hexdigest()[:10]
    newest_hdr = max(os.path.getmtime(p) for p in HEADERS)
    jobs, objs = [], []
    for src in sources():
        obj = os.path.join(objdir, f"{os.path.splitext(os.path.basename(src))[0]}.{tag}.o")
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(newest_hdr, os.path.getmtime(src)):
            jobs.append([nvcc()] + NVCC_FLAGS + list(extra) + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src])
    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            list(ex.map(subprocess.check_call, jobs))
    if jobs or not os.path.exists(lib) or os.path.getmtime(lib) < max(os.path.getmtime(o) for o in objs):
        tmp = f"{lib}.{os.getpid()}.tmp"
        subprocess.check_call([nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + objs)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
