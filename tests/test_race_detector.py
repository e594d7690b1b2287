"""The race-detector build of the host model (tests/emu/race_check.py): it must find the race that a removed
barrier opens, and report nothing on the kernels as they are.  Small cases only; the long runs are in profiles/."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SCRIPT = os.path.join(ROOT, "tests", "emu", "race_check.py")


def _libtsan():
    try:
        path = subprocess.check_output(["gcc", "-print-file-name=libtsan.so"], text=True).strip()
    except (OSError, subprocess.CalledProcessError):
        return None
    return path if os.path.isabs(path) and os.path.exists(path) else None


pytestmark = pytest.mark.skipif(_libtsan() is None, reason="gcc's libtsan is not installed")


def test_the_detector_finds_the_race_that_a_removed_barrier_opens():
    out = subprocess.run([sys.executable, SCRIPT, "--self-test"], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stdout[-3000:] + out.stderr[-2000:]
    assert "the detector found the opened race" in out.stdout


def test_no_report_on_the_kernels_as_they_are():
    out = subprocess.run([sys.executable, SCRIPT, "-k", "test_configs_bit_exact and 0-1 or test_frontend_slice and 10ns or test_refit_tracks and 1-12"],
                         capture_output=True, text=True, timeout=1500, cwd=ROOT)
    assert out.returncode == 0, out.stdout[-3000:] + out.stderr[-2000:]
    assert "ThreadSanitizer reports: 0" in out.stdout
