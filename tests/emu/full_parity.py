"""Parity of the kernels in the host model at (or towards) the BASELINE configs' full sizes -- a long-running companion of
tests/test_emulated_kernels.py, not part of the pytest suite.  TEST INFRASTRUCTURE.

    python tests/emu/full_parity.py --cfg 1 --events 1000 [--first 0] [--chunk 50] [--procs 8] [--hits-idx H --grid-idx G]

Every event goes through hough_vote (digest), hough_find_clusters and hough_assign_hits of tests/emu/libhough_emu.so and is
compared with oracle/hough_oracle.c: digests, n_found, every kept record (bytes), every label.  Prints one summary line.
"""
import argparse
import multiprocessing as mp
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, os.path.join(ROOT, "tests"), HERE):
    if p not in sys.path:
        sys.path.insert(0, p)


def work(job):
    cfg, hi, gi, first, n = job
    import hough_emu as E
    from oracle import hough_c as C
    from paper_2511_02742_b200 import synth
    from util import params_of
    wl = synth.workload(cfg, hi, gi)
    b = synth.generate(wl, first, n)
    p = params_of(wl)
    dt = E.HOUGH_U16 if wl.count_dtype == "u16" else E.HOUGH_I32
    g = E.run(p, b.u, b.v, b.offsets, dt, want_acc=False)
    o = C.run_batch(b.u, b.v, b.offsets, p, want_digest=True)
    bad = []
    if g["emu_violations"] or g["bounds_violations"] or g["status"]:
        bad.append(f"violations emu={g['emu_violations']} bounds={g['bounds_violations']} status={g['status']}")
    if not (g["digest"] == o["digest"]).all():
        bad.append("digest")
    if not (g["n_found"] == o["n_found"]).all():
        bad.append("n_found")
    if not (g["labels"] == o["labels"]).all():
        bad.append("labels")
    for e in range(n):
        k = min(int(o["n_found"][e]), p.max_candidates)
        if g["cands"][e, :k].tobytes() != o["cands"][e, :k].tobytes():
            bad.append(f"records of event {first + e}")
            break
    return dict(first=first, n=n, hits=int(b.n_hits), deferred=g["deferred"], fast=g["info"]["fast_groups"], bad=bad,
                n_found_max=int(o["n_found"].max()) if n else 0)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg", type=int, required=True)
    ap.add_argument("--hits-idx", type=int, default=0)
    ap.add_argument("--grid-idx", type=int, default=0)
    ap.add_argument("--first", type=int, default=0)
    ap.add_argument("--events", type=int, required=True)
    ap.add_argument("--chunk", type=int, default=50)
    ap.add_argument("--procs", type=int, default=max(1, (os.cpu_count() or 2) - 1))
    a = ap.parse_args()
    import hough_emu as E
    E.lib()                                                       # build once, before the workers start
    jobs = [(a.cfg, a.hits_idx, a.grid_idx, f, min(a.chunk, a.first + a.events - f)) for f in range(a.first, a.first + a.events, a.chunk)]
    t0 = time.time()
    with mp.get_context("spawn").Pool(a.procs) as pool:
        res = pool.map(work, jobs, chunksize=1)
    bad = [(r["first"], r["bad"]) for r in res if r["bad"]]
    print(f"cfg {a.cfg} (hits_idx {a.hits_idx}, grid_idx {a.grid_idx}) events [{a.first}, {a.first + a.events}): "
          f"{sum(r['hits'] for r in res)} hits, fast_groups {res[0]['fast']}, deferred {sum(r['deferred'] for r in res)}, "
          f"largest n_found {max(r['n_found_max'] for r in res)}, {time.time() - t0:.0f} s on {a.procs} processes: "
          + ("ALL IDENTICAL (digests, n_found, records, labels; no violation)" if not bad else f"MISMATCH {bad[:5]}"))
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
