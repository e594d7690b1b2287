import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_addoption(parser):
    parser.addoption("--hough-variant", action="store", default="",
                     help="run the GPU tests against a debug variant of the library (bounds | timers); see DESIGN.md 'GPU gate'")
    parser.addoption("--gate", action="store_true", default=False,
                     help="only the small gate cases (<= 8 events each), for the bounds build and compute-sanitizer runs")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: longer CPU test")
    config.addinivalue_line("markers", "gate: small GPU case that is safe to run first on an untested build")
    variant = config.getoption("--hough-variant")
    if variant:
        from paper_2511_02742_b200 import build, hough
        hough.load_library(build.build(variant=variant))
    else:
        # a fresh checkout has no libhough.so (built artefacts are not in the history): build it now if it is missing or older than
        # its sources -- a no-op otherwise.  Without nvcc nothing is built, and the binding still fails loudly when a test loads it.
        try:
            from paper_2511_02742_b200 import build
            build.build()
        except Exception as exc:  # noqa: BLE001
            print(f"conftest: libhough.so was not (re)built: {exc}", file=sys.stderr)


def pytest_collection_modifyitems(config, items):
    if config.getoption("--gate"):
        skip = pytest.mark.skip(reason="not a gate case")
        for it in items:
            if "gate" not in it.keywords:
                it.add_marker(skip)
    # small before large: among the GPU tests the gate cases (<= 8 events each) run first, so that under -x a build
    # that is wrong fails on a handful of events before anything is launched at full size.  The sort is stable: everything else
    # (and every CPU test) keeps its place relative to its peers.
    gpu_positions = [i for i, it in enumerate(items) if "gpu" in it.keywords]
    gpu_items = sorted((items[i] for i in gpu_positions), key=lambda it: 0 if "gate" in it.keywords else 1)
    for i, it in zip(gpu_positions, gpu_items):
        items[i] = it
