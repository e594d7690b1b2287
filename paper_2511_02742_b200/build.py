"""Build step of libhough.so: nvcc, sm_100a only, in-tree (the .so travels to the GPU box with the snapshot).

    python -m paper_2511_02742_b200.build [--force] [--verbose]

The library is plain CUDA runtime + C ABI (include/hough.h); nothing here links against torch.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
SOURCES = [os.path.join(_HERE, "csrc", "hough_lib.cu")]
DEPENDS = SOURCES + [os.path.join(_HERE, "csrc", "hough_kernels.cuh"), os.path.join(_HERE, "csrc", "hough_fast.cuh"), os.path.join(_ROOT, "include", "hough.h")]
LIB = os.path.join(_HERE, "libhough.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--use_fast_math",
              "-Xcompiler", "-fPIC,-O2,-Wall", "-shared", "-cudart", "static"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPENDS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    extra = os.environ.get("HOUGH_NVCC_EXTRA", "").split()      # e.g. -DHOUGH_PHASE_TIMERS for the diagnostic build
    cmd = [nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
