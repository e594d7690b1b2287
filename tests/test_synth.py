"""The seeded input generator: reproducible, shaped as BASELINE.json's configs say."""
import numpy as np
import pytest

from paper_2511_02742_b200 import synth
from util import read_golden_table


def test_golden_sha256():
    for cfg, hi, gi, first, n, n_hits, sha in read_golden_table("synth_sha256.txt"):
        b = synth.generate(synth.workload(int(cfg), int(hi), int(gi)), int(first), int(n))
        assert b.n_hits == int(n_hits) and b.sha256() == sha


def test_shapes_follow_baseline_configs():
    b0 = synth.generate(synth.workload(0))
    assert b0.n_events == 1 and b0.n_hits == 158                       # 3*48 + round(0.1*144)
    b1 = synth.generate(synth.workload(1), 0, 100)
    assert (np.diff(b1.offsets) == 288).all()                           # 5*48 + 48
    b2 = synth.generate(synth.workload(2), 0, 200)
    n2 = np.diff(b2.offsets)
    ntr = np.diff(b2.track_offsets)
    assert ntr.min() >= 10 and ntr.max() <= 20 and 600 < n2.mean() < 1200
    b3 = synth.generate(synth.workload(3), 0, 20)
    n3 = np.diff(b3.offsets)
    assert 2700 < n3.mean() < 2870 and n3.max() <= 2880                 # 1920*0.95 + 960
    for hi, h in enumerate(synth.CFG4_HITS):
        b4 = synth.generate(synth.workload(4, hi, 0), 0, 5)
        assert (np.diff(b4.offsets) == h).all()
    for b in (b0, b1, b2, b3):
        assert b.u.dtype == np.float32 and b.v.dtype == np.float32 and b.offsets.dtype == np.int64
        assert np.abs(b.u).max() <= 94.0 and np.abs(b.v).max() < 256.0
        # every vote stays inside rho in [-256, 256): max |rho| = hypot(94, 194 + smear)
        assert np.hypot(b.u.astype(np.float64), b.v.astype(np.float64)).max() < 255.0


def test_slicing_is_consistent_across_chunks():
    wl = synth.workload(2)
    a = synth.generate(wl, 995, 10)                                     # straddles the chunk boundary at 1000
    b = synth.generate(wl, 990, 20)
    s = b.slice(5, 15)
    assert (a.u == s.u).all() and (a.v == s.v).all() and (a.offsets == s.offsets).all()
    assert a.first_event == 995 and (a.truth_track == s.truth_track).all()


def test_track_hits_lie_on_their_lines():
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 3)
    for e in range(3):
        u, v = b.event(e)
        tt = b.truth_track[b.offsets[e]:b.offsets[e + 1]]
        for k in range(5):
            m, c = b.track_m[b.track_offsets[e] + k], b.track_c[b.track_offsets[e] + k]
            sel = tt == k
            assert sel.sum() == 48
            assert np.abs(v[sel] - (m * u[sel] + c)).max() < 0.6        # 0.1 mm smearing, < 6 sigma
        assert (tt == -1).sum() == 48
