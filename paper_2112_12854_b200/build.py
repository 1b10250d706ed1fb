"""In-tree build of libep.so (the C-ABI library of include/ep.h) with nvcc for sm_100a.

    python -m paper_2112_12854_b200.build [--force] [-v]

nvcc cross-compiles without a GPU; the static CUDA runtime is linked so the library loads on a machine without a
driver (every compute entry point then returns EP_ERR_CUDA).  The .so is git-ignored but travels with the tree.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libep.so")
SOURCES = ["ep_api.cu", "ep_kernels.cu", "ep_elliptic.cu", "ep_noalloc.cu", "ep_host.cpp"]
HEADERS = ["ep_host.h", "ep_kernels.cuh", "ep_math.cuh", "ep_tp06.cuh", "ep_crn98.cuh", "ep_stewart.cuh", os.path.join("..", "..", "include", "ep.h")]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libep cannot be built (there is no CPU fallback)")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.exists(d) and os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale()):
        return LIB
    cmd = [_nvcc(), "-O3", "-std=c++20", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC,-O2", "-shared", "-cudart", "static"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
