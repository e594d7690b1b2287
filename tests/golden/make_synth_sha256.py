"""Writes tests/golden/synth_sha256.txt: SHA-256 of generated input arrays (u || v || offsets) of small slices of
every workload.  Calls only the input generator (paper_2511_02742_b200/synth.py), nothing from the CUDA path.
Run from the repo root:  python tests/golden/make_synth_sha256.py"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from paper_2511_02742_b200 import synth  # noqa: E402

SLICES = [(0, 0, 0, 0, 1), (1, 0, 0, 0, 1000), (2, 0, 0, 0, 50), (2, 0, 0, 9990, 10), (3, 0, 0, 0, 10), (3, 0, 0, 99995, 5),
          (4, 0, 0, 0, 20), (4, 1, 1, 0, 20), (4, 2, 2, 1000, 10), (4, 3, 3, 49990, 10)]

if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "synth_sha256.txt")
    with open(out, "w") as f:
        f.write("# SHA-256 of (u || v || offsets) bytes of synth.generate(workload(cfg, hits_idx, grid_idx), first, n).\n")
        f.write("# Written by tests/golden/make_synth_sha256.py (input generator only). Recipe: DESIGN.md 'Input recipe'.\n")
        f.write("# columns: cfg hits_idx grid_idx first_event n_events n_hits sha256\n")
        for cfg, hi, gi, first, n in SLICES:
            b = synth.generate(synth.workload(cfg, hi, gi), first, n)
            f.write(f"{cfg} {hi} {gi} {first} {n} {b.n_hits} {b.sha256()}\n")
    print(open(out).read())
