"""Build step of tests/emu/libhough_emu.so: the kernel and host sources of paper_2511_02742_b200/csrc compiled with g++ for
the host CUDA model of cuda_emu.h.  TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT (nothing under paper_2511_02742_b200/
imports or loads it).

    python tests/emu/build_emu.py [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(os.path.dirname(_HERE))
_CSRC = os.path.join(_ROOT, "paper_2511_02742_b200", "csrc")
LIB = os.path.join(_HERE, "libhough_emu.so")
DEPENDS = [os.path.join(_HERE, "cuda_emu.h"), os.path.join(_HERE, "cuda_emu.cpp"), os.path.join(_ROOT, "include", "hough.h")] + \
          [os.path.join(_CSRC, f) for f in sorted(os.listdir(_CSRC))]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(d) <= os.path.getmtime(LIB) for d in DEPENDS):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    # -DHOUGH_BOUNDS: the kernels' own index checks are compiled in as well (a failed check is reported, not performed)
    cmd = ["g++", "-std=c++17", "-O2", "-g", "-fPIC", "-shared", "-ffp-contract=off", "-fno-strict-aliasing", "-DHOUGH_EMU", "-DHOUGH_BOUNDS",
           "-Wall", "-Wno-unused-function", "-Wno-unused-variable", "-Wno-unknown-pragmas", "-Wno-sign-compare",
           "-I", _HERE, "-x", "c++", os.path.join(_CSRC, "hough_lib.cu"), os.path.join(_HERE, "cuda_emu.cpp"), "-o", tmp, "-pthread"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
