"""Dry run of bench.py against the host model: `python tests/emu/bench_dry.py [bench.py arguments]`.  TEST INFRASTRUCTURE.

It checks that the benchmark's own code path (plan, warm-up, timed loop, end-to-end leg through hough_run_host, roofline and
cpu_baseline objects, --all-configs) executes and prints a well-formed line on a machine without a GPU.  CUDA events become a
counter and the live peak measurement a constant, so EVERY NUMBER IT PRINTS IS MEANINGLESS; only the structure of the line and
the two parity flags in it (`gpu_outputs_identical_on_sample`, `e2e.same_as_device_results`) mean anything.
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for _p in (HERE, ROOT, os.path.join(ROOT, "tests")):
    if _p not in sys.path:
        sys.path.insert(0, _p)

import torch  # noqa: E402
import emu_plugin  # noqa: E402,F401  (points the binding at the host-model library, "cuda" devices at the CPU)
from paper_2511_02742_b200 import hough as H  # noqa: E402


class FakeEvent:
    n = 0

    def __init__(self, enable_timing=False):
        self.t = None

    def record(self, stream=None):
        FakeEvent.n += 1
        self.t = FakeEvent.n

    def elapsed_time(self, other):
        return float(other.t - self.t)


torch.cuda.set_device = lambda *a, **k: None
torch.cuda.Event = FakeEvent
H.hough_measure_smem_atomic_peak = lambda dev, ms: (1.0e12, 1000.0)

if __name__ == "__main__":
    import bench
    sys.exit(bench.main())
