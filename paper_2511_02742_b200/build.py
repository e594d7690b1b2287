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
# every file of csrc/ (hough_lib.cu includes all the .cuh headers) and the public header
DEPENDS = sorted(os.path.join(_HERE, "csrc", f) for f in os.listdir(os.path.join(_HERE, "csrc"))) + [os.path.join(_ROOT, "include", "hough.h")]
LIB = os.path.join(_HERE, "libhough.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-O2,-Wall", "-shared", "-cudart", "static"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


# Debug variants: same sources, one extra define, their own file next to libhough.so.
#   bounds  -DHOUGH_BOUNDS        every computed index inside the kernels is range-checked; a failed check sets
#                                 HOUGH_STATUS_INTERNAL and skips the access (nothing is stored out of range, nothing traps)
#   timers  -DHOUGH_PHASE_TIMERS  per-phase SM-cycle sums (hough_plan_debug_counters)
VARIANTS = {"": [], "bounds": ["-DHOUGH_BOUNDS"], "timers": ["-DHOUGH_PHASE_TIMERS"]}


def lib_path(variant: str = "") -> str:
    return LIB if not variant else os.path.join(_HERE, f"libhough_{variant}.so")


def is_stale(variant: str = "") -> bool:
    lib = lib_path(variant)
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in DEPENDS)


def build(force: bool = False, verbose: bool = False, variant: str = "") -> str:
    lib = lib_path(variant)
    if not force and not is_stale(variant):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [nvcc()] + NVCC_FLAGS + VARIANTS[variant] + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    subprocess.check_call(cmd)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    var = ""
    for a in sys.argv[1:]:
        if a.startswith("--variant="):
            var = a.split("=", 1)[1]
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, variant=var))
