"""Build step of tests/emu/libhough_emu.so: the kernel and host sources of paper_2511_02742_b200/csrc compiled with g++ for
the host CUDA model of cuda_emu.h.  TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT (nothing under paper_2511_02742_b200/
imports or loads it).

    python tests/emu/build_emu.py [--force] [--tsan | --ubsan | --no-bounds]

--tsan builds tests/emu/libhough_emu_tsan.so, the race-detector variant: the kernel sources are compiled with
-fsanitize=thread and -DHOUGH_EMU_TSAN (every CUDA thread a ThreadSanitizer fiber, see cuda_emu.cpp); the model itself
(cuda_emu.cpp) is NOT instrumented, so the detector sees the kernels' memory accesses and only the synchronisation CUDA
defines.  Load it in a process started with LD_PRELOAD=$(gcc -print-file-name=libtsan.so); tests/emu/race_check.py does.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(os.path.dirname(_HERE))
_CSRC = os.path.join(_ROOT, "paper_2511_02742_b200", "csrc")
LIB = os.path.join(_HERE, "libhough_emu.so")
LIB_TSAN = os.path.join(_HERE, "libhough_emu_tsan.so")
DEPENDS = [os.path.join(_HERE, "cuda_emu.h"), os.path.join(_HERE, "cuda_emu.cpp"), os.path.join(_ROOT, "include", "hough.h")] + \
          [os.path.join(_CSRC, f) for f in sorted(os.listdir(_CSRC))]


def build_tsan(force: bool = False, csrc: str = _CSRC, out: str = LIB_TSAN) -> str:
    """csrc / out: race_check.py --self-test builds a copy of the sources with one barrier taken out."""
    if not force and csrc == _CSRC and os.path.exists(out) and all(os.path.getmtime(d) <= os.path.getmtime(out) for d in DEPENDS):
        return out
    tmp = out + f".tmp{os.getpid()}"
    common = ["g++", "-std=c++17", "-O1", "-g", "-fPIC", "-ffp-contract=off", "-fno-strict-aliasing", "-DHOUGH_EMU", "-DHOUGH_EMU_TSAN",
              "-DHOUGH_BOUNDS", "-Wno-unknown-pragmas", "-I", _HERE]
    obj_model, obj_kernels = tmp + ".model.o", tmp + ".kernels.o"
    try:
        subprocess.check_call(common + ["-c", os.path.join(_HERE, "cuda_emu.cpp"), "-o", obj_model])
        subprocess.check_call(common + ["-fsanitize=thread", "-c", "-x", "c++", os.path.join(csrc, "hough_lib.cu"), "-o", obj_kernels])
        subprocess.check_call(["g++", "-shared", "-fsanitize=thread", obj_kernels, obj_model, "-o", tmp, "-pthread"])
    finally:
        for o in (obj_model, obj_kernels):
            if os.path.exists(o):
                os.remove(o)
    os.replace(tmp, out)
    return out


LIB_UBSAN = os.path.join(_HERE, "libhough_emu_ubsan.so")
LIB_NOBOUNDS = os.path.join(_HERE, "libhough_emu_nobounds.so")


def build_nobounds(force: bool = False) -> str:
    """The host model WITHOUT -DHOUGH_BOUNDS: the kernels exactly as the product compiles them (the HB() checks are gone), with
    only the model's guard pages and shared-window checks left.  An access that only HB() kept in range would fault here.
    Use with HOUGH_EMU_LIB=tests/emu/libhough_emu_nobounds.so."""
    if not force and os.path.exists(LIB_NOBOUNDS) and all(os.path.getmtime(d) <= os.path.getmtime(LIB_NOBOUNDS) for d in DEPENDS):
        return LIB_NOBOUNDS
    tmp = LIB_NOBOUNDS + f".tmp{os.getpid()}"
    subprocess.check_call(["g++", "-std=c++17", "-O2", "-g", "-fPIC", "-shared", "-ffp-contract=off", "-fno-strict-aliasing", "-DHOUGH_EMU",
                           "-Wno-unknown-pragmas", "-I", _HERE, "-x", "c++", os.path.join(_CSRC, "hough_lib.cu"),
                           os.path.join(_HERE, "cuda_emu.cpp"), "-o", tmp, "-pthread"])
    os.replace(tmp, LIB_NOBOUNDS)
    return LIB_NOBOUNDS


def build_ubsan(force: bool = False) -> str:
    """The host model with -fsanitize=undefined: shift counts >= the width (x86 masks them, the GPU clamps them -- a place
    where the model and the hardware would silently differ), signed overflow, misaligned vector accesses.  Run with
    LD_PRELOAD=$(gcc -print-file-name=libubsan.so) HOUGH_EMU_LIB=tests/emu/libhough_emu_ubsan.so UBSAN_OPTIONS=log_path=..."""
    if not force and os.path.exists(LIB_UBSAN) and all(os.path.getmtime(d) <= os.path.getmtime(LIB_UBSAN) for d in DEPENDS):
        return LIB_UBSAN
    tmp = LIB_UBSAN + f".tmp{os.getpid()}"
    subprocess.check_call(["g++", "-std=c++17", "-O1", "-g", "-fPIC", "-shared", "-ffp-contract=off", "-fno-strict-aliasing", "-DHOUGH_EMU",
                           "-DHOUGH_BOUNDS", "-fsanitize=undefined,float-cast-overflow", "-fno-sanitize=vptr", "-Wno-unknown-pragmas", "-I", _HERE, "-x", "c++",
                           os.path.join(_CSRC, "hough_lib.cu"), os.path.join(_HERE, "cuda_emu.cpp"), "-o", tmp, "-pthread"])
    os.replace(tmp, LIB_UBSAN)
    return LIB_UBSAN


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
    which = build_tsan if "--tsan" in sys.argv else build_ubsan if "--ubsan" in sys.argv else build_nobounds if "--no-bounds" in sys.argv else build
    print(which(force="--force" in sys.argv))
