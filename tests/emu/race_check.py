"""Data-race check of the kernels in the host model under ThreadSanitizer.  TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT;
a long-running companion of tests/test_emulated_kernels.py, not part of the pytest suite.

    python tests/emu/race_check.py [-k PYTEST_EXPRESSION] [--all] [--keep-logs DIR]
    python tests/emu/race_check.py --self-test       # the detector must FIND the race that a removed barrier opens
    python tests/emu/race_check.py --fuzz N --seed S # N random plans of tests/emu/fuzz_parity.py instead of the pytest cases

Builds tests/emu/libhough_emu_tsan.so (build_emu.py --tsan: the kernel sources compiled with -fsanitize=thread, every CUDA thread
a detector fiber, the only happens-before edges inside a CTA being __syncthreads, __syncwarp and program order; atomics relaxed)
and runs cases of tests/test_emulated_kernels.py against it in a child process that has libtsan preloaded.  The cases keep their
parity assertions, so a run is "checked" only if the results are also identical to the oracle's.  Prints the number of
detector reports (0 expected) and the first few; exit code 1 if there is a report or a case fails.

What it can and cannot show: a report is two accesses to one address from two CUDA threads, at least one a plain write, with
no barrier / __syncwarp / atomic-free ordering between them IN THE SCHEDULE THAT RAN (the detector is dynamic).  The lock-free
union-find (uf_* / suf_*: path halving with plain loads next to atomicCAS / atomicMin on the same words, benign by design,
DESIGN.md Sec. 7) is suppressed by function name in race_check.supp.  It says nothing about the hardware memory model.
"""
from __future__ import annotations

import argparse
import glob
import os
import re
import shutil
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))

# one case per kernel and per hand-over path; the whole file takes about ten times longer
DEFAULT_K = ("test_configs_bit_exact and (0-1 or 2-12 or 3-6) or test_concurrent_ctas or test_mixed_batch or test_refit_tracks "
             "or test_frontend_slice or test_frontend_feeds or test_peeloff_variant or test_two_stage_variant "
             "or test_dense_workload or test_edge_set_as_one_ragged_batch or test_run_host_chunked or test_theta_wrap_variant "
             "or test_theta_wrap_does_not")


BARRIER = "__syncthreads();  // all votes of the strip are in"


def sources_without_the_vote_barrier(tmp: str) -> str:
    """A copy of the kernel sources in which the barrier between the votes and the scan of a strip is missing (both Hough
    kernels): scanning threads then read counters that other threads still add to."""
    csrc = os.path.join(tmp, "pkg", "csrc")
    shutil.copytree(os.path.join(ROOT, "paper_2511_02742_b200", "csrc"), csrc)
    shutil.copytree(os.path.join(ROOT, "include"), os.path.join(tmp, "include"))
    dropped = 0
    for name in ("hough_fast.cuh", "hough_kernels.cuh"):
        path = os.path.join(csrc, name)
        text = open(path).read()
        dropped += text.count(BARRIER)
        open(path, "w").write(text.replace(BARRIER, "/* barrier removed by race_check.py --self-test */"))
    assert dropped == 2, "the barrier comment that --self-test looks for has changed"
    return csrc


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("-k", default=DEFAULT_K)
    ap.add_argument("--all", action="store_true", help="every case of tests/test_emulated_kernels.py")
    ap.add_argument("--keep-logs", default=None)
    ap.add_argument("--self-test", action="store_true")
    ap.add_argument("--fuzz", type=int, default=0, help="run this many cases of fuzz_parity.py under the detector instead")
    ap.add_argument("--seed", type=int, default=1)
    args = ap.parse_args()
    sys.path.insert(0, HERE)
    import build_emu
    which = "tsan"
    if args.self_test:
        tmp = tempfile.mkdtemp(prefix="hough_tsan_selftest_")
        which = build_emu.build_tsan(force=True, csrc=sources_without_the_vote_barrier(tmp), out=os.path.join(tmp, "libhough_emu_tsan_nobarrier.so"))
        args.k, args.all = "test_configs_bit_exact and 0-1 and not small_lists", False
    else:
        build_emu.build_tsan()
    libtsan = subprocess.check_output(["gcc", "-print-file-name=libtsan.so"], text=True).strip()
    libtsan = os.path.realpath(libtsan)
    logdir = args.keep_logs or tempfile.mkdtemp(prefix="hough_tsan_")
    os.makedirs(logdir, exist_ok=True)
    opts = ["suppressions=" + os.path.join(HERE, "race_check.supp"), "log_path=" + os.path.join(logdir, "tsan"), "halt_on_error=0",
            "exitcode=0", "report_signal_unsafe=0", "report_thread_leaks=0", "second_deadlock_stack=0", "detect_deadlocks=0"]
    env = dict(os.environ, LD_PRELOAD=libtsan, HOUGH_EMU_LIB=which, TSAN_OPTIONS=":".join(opts), OMP_NUM_THREADS="1",
               OPENBLAS_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_emulated_kernels.py"), "-q", "-p", "no:cacheprovider"]
    if args.fuzz:
        cmd = [sys.executable, os.path.join(HERE, "fuzz_parity.py"), "--cases", str(args.fuzz), "--seed", str(args.seed)]
    elif not args.all:
        cmd += ["-k", args.k]
    rc = subprocess.call(cmd, env=env, cwd=ROOT)
    reports, first = 0, []
    for path in sorted(glob.glob(os.path.join(logdir, "tsan.*"))):
        text = open(path, errors="replace").read()
        for block in re.split(r"(?m)^==================\n", text):
            if "WARNING: ThreadSanitizer" in block:
                reports += 1
                if len(first) < 3:
                    first.append("\n".join(block.splitlines()[:14]))
    print(f"race_check: exit code of the cases {rc}; ThreadSanitizer reports: {reports}; logs: {logdir}")
    for b in first:
        print("----\n" + b)
    if args.self_test:
        print("race_check --self-test: " + ("the detector found the opened race" if reports else "NO REPORT: the detector is blind"))
        return 0 if reports else 1
    return 1 if (rc != 0 or reports) else 0


if __name__ == "__main__":
    sys.exit(main())
