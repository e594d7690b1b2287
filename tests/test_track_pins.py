"""Pins of the oracle stages around the Hough core (oracle/track_def.py: O9 refit, O10 found criterion, O11 time slicing,
O12 CORDIC phi, O13 peel-off) against what the mathematics fixes: closed forms, library routines, error bounds, brute force.
No GPU, no product code."""
import math

import numpy as np
import pytest

from oracle import hough_def as D
from oracle import track_def as T
from paper_2511_02742_b200 import synth
from util import std_params

FE = T.FrontEnd()


# ----------------------------------------------------------------------------- O12 CORDIC phi
def test_cordic_table_values():
    A = T.cordic_table(FE)
    assert A[0] == 45 * 65536                                   # atan(1) = 45 degrees exactly
    assert A[1] == round(26.56505117707799 * 65536)             # atan(1/2), textbook value
    assert all(A[i] > A[i + 1] > 0 for i in range(len(A) - 1))
    assert abs(A[10] / 65536 - math.degrees(2.0 ** -10)) < 1e-4  # small angles: atan(x) ~ x


def test_cordic_equals_atan2_within_the_derived_bound():
    rng = np.random.default_rng(7)
    worst = 0.0
    pts = [(int(a), int(b)) for a, b in rng.integers(-32768, 32769, (4000, 2))]
    pts += [(int(r * math.cos(a)), int(r * math.sin(a))) for r in (4480, 18560) for a in np.linspace(-math.pi, math.pi, 721)]
    pts += [(1, 0), (0, 1), (-1, 0), (0, -1), (1, 1), (-1, 1), (-1, -1), (1, -1), (32768, 1), (-32768, 1), (-32768, -1), (3, -32768)]
    for xq, yq in pts:
        if (xq, yq) == (0, 0):
            continue
        phi = T.cordic_phi_q(xq, yq, FE) / 65536.0
        ref = math.degrees(math.atan2(yq, xq))
        err = abs(phi - ref)
        err = min(err, abs(err - 360.0))                         # the branch cut at +-180
        bound = T.cordic_error_bound_deg(math.hypot(xq, yq), FE)
        assert err <= bound, (xq, yq, phi, ref, bound)
        if math.hypot(xq, yq) >= 4480:
            worst = max(worst, err)
    assert worst < 5e-4                                          # detector radii (>= 70 mm): well below the 0.15 degree strip pitch


def test_cordic_reflection_in_x_is_exact():
    rng = np.random.default_rng(8)
    for xq, yq in rng.integers(1, 30000, (300, 2)):
        xq, yq = int(xq), int(yq)
        a = T.cordic_phi_q(xq, yq, FE)
        assert T.cordic_phi_q(-xq, yq, FE) == 180 * 65536 - a
        b = T.cordic_phi_q(xq, -yq, FE)
        assert T.cordic_phi_q(-xq, -yq, FE) == -180 * 65536 - b


def test_cordic_is_monotone_along_a_circle():
    r = 12000
    prev = None
    for a in np.linspace(-179.0, 179.0, 2000):
        xq, yq = round(r * math.cos(math.radians(a))), round(r * math.sin(math.radians(a)))
        phi = T.cordic_phi_q(xq, yq, FE)
        if prev is not None:
            assert phi >= prev - 40                              # 40 LSB = 6e-4 degree of slack for the iteration residue
        prev = phi


def test_cordic_state_stays_in_int32_for_the_largest_inputs():
    for xq, yq in ((32768, 32768), (-32768, 32768), (32768, -32768), (0, 32768), (32768, 0), (1, -32768)):
        T.cordic_phi_q(xq, yq, FE)                               # asserts inside


# ----------------------------------------------------------------------------- O11 time slicing
def brute_windows(t, fe):
    """Window membership straight from the inequality t0 + w step <= t < t0 + w step + width, on times rounded to 2^-8 ns."""
    tq = round(float(np.float32(t)) * 256)
    return [w for w in range(fe.windows_per_fill) if round(fe.t0 * 256) + w * round(fe.step * 256) <= tq < round(fe.t0 * 256) + w * round(fe.step * 256) + round(fe.width * 256)]


def test_slice_membership_equals_the_window_inequality():
    rng = np.random.default_rng(9)
    fe = T.FrontEnd(t0=3.0, windows_per_fill=9)
    n = 400
    t = np.concatenate([rng.uniform(-12, 70, n - 8), [3.0, 8.0, 13.0, 12.99609375, 2.99609375, 48.0, 52.99609375, 53.0]]).astype(np.float32)
    x = rng.uniform(70, 290, n).astype(np.float32); y = rng.uniform(-290, 290, n).astype(np.float32)
    z = rng.uniform(-200, 200, n).astype(np.float32)
    u, v, src, counts = T.slice_fill(x, y, z, t, fe)
    pos = 0
    for w in range(fe.windows_per_fill):
        members = [i for i in range(n) if w in brute_windows(t[i], fe)]
        got = src[pos:pos + counts[w]]
        assert list(got) == members                               # B4: input order inside a window
        np.testing.assert_array_equal(v[pos:pos + counts[w]], z[members])
        pos += counts[w]
    assert pos == len(src)
    # 10 ns windows every 5 ns: an interior hit is in exactly two windows
    interior = [i for i in range(n) if 3.0 + 5.0 <= t[i] < 3.0 + 5.0 * 9]
    assert all(len(brute_windows(t[i], fe)) == 2 for i in interior)
    # window edges are half open
    assert brute_windows(np.float32(8.0), fe) == [0, 1] and brute_windows(np.float32(13.0), fe) == [1, 2]
    assert brute_windows(np.float32(2.99609375), fe) == [] and brute_windows(np.float32(3.0), fe) == [0]


def test_slice_drops_invalid_hits_and_maps_phi():
    fe = T.FrontEnd(windows_per_fill=2)
    x = np.array([100.0, np.nan, 0.0, 600.0, 0.0, -100.0, 100.0], np.float32)
    y = np.array([0.0, 1.0, 0.0, 0.0, 100.0, 0.0, 100.0], np.float32)
    z = np.array([1.0, 2.0, 3.0, 4.0, 5.0, 6.0, np.inf], np.float32)
    t = np.full(7, 6.0, np.float32)
    u, v, src, counts = T.slice_fill(x, y, z, t, fe)
    assert list(counts) == [3, 3] and list(src) == [0, 4, 5, 0, 4, 5]     # NaN, origin, out-of-range and Inf hits are in no window
    assert abs(u[0]) < 1e-3 and abs(u[1] - 90.0) < 1e-3 and abs(abs(u[2]) - 180.0) < 1e-3
    assert u.dtype == np.float32 and all(float(a) * 65536 == round(float(a) * 65536) for a in u)   # phi_q 2^-16 is exact in fp32


def test_slice_batch_offsets_and_global_indices():
    rng = np.random.default_rng(10)
    fe = T.FrontEnd(windows_per_fill=4)
    n = 90
    x, y, z = (rng.uniform(-290, 290, n).astype(np.float32) for _ in range(3))
    t = rng.uniform(0, 25, n).astype(np.float32)
    fo = np.array([0, 30, 30, 90], np.int64)
    u, v, src, offsets = T.slice_batch(x, y, z, t, fo, fe)
    assert len(offsets) == 3 * 4 + 1 and offsets[-1] == len(u)
    assert (offsets[4:9] == offsets[4]).all()                             # the empty fill has four empty windows
    assert ((src[: offsets[4]] < 30).all()) and ((src[offsets[8]:] >= 30).all())
    np.testing.assert_array_equal(v, z[src])


# ----------------------------------------------------------------------------- O9 / O10 refit and found criterion
GEOM = T.PlaneGeometry(origin=-94.0, pitch=4.0, n_planes=48)


def test_refit_recovers_an_exact_line():
    p = std_params(256, 256)
    uu, _ = synth.ideal_track(0.0, 0.0)
    m, c = 0.375, -12.25                                                  # v = m u + c is a multiple of 1/64 at every plane
    vv = (m * uu.astype(np.float64) + c).astype(np.float32)
    fits = T.refit_event(uu, vv, np.zeros(48, np.int32), 1, p, GEOM)
    f = fits[0]
    assert f.n_hits == 48 and f.plane_mask == 2 ** 48 - 1 and f.max_run == 48 and f.flags == T.FIT_FOUND
    assert float(f.slope) == m and float(f.intercept) == c


def test_refit_equals_numpy_polyfit_on_the_quantised_hits():
    rng = np.random.default_rng(11)
    p = std_params(256, 256)
    n = 300
    u = rng.uniform(-94, 94, n).astype(np.float32); v = rng.uniform(-194, 194, n).astype(np.float32)
    labels = rng.integers(-1, 5, n).astype(np.int32)
    fits = T.refit_event(u, v, labels, 5, p, GEOM)
    uq, vq = np.round(u.astype(np.float64) * 64) / 64, np.round(v.astype(np.float64) * 64) / 64
    for s in range(5):
        sel = labels == s
        m, c = np.polyfit(uq[sel], vq[sel], 1)
        assert fits[s].n_hits == int(sel.sum())
        assert abs(float(fits[s].slope) - m) <= 1e-6 * max(1.0, abs(m)) and abs(float(fits[s].intercept) - c) <= 1e-5 * max(1.0, abs(c))
    # permuting the hits changes nothing: the sums are exact integers
    pm = rng.permutation(n)
    assert T.refit_event(u[pm], v[pm], labels[pm], 5, p, GEOM) == fits


def test_refit_two_points_and_degenerate_cases():
    p = std_params(256, 256)
    u = np.array([-10.0, 30.0, 5.0, 5.0, 7.0], np.float32); v = np.array([2.0, 12.0, 1.0, 9.0, 3.0], np.float32)
    labels = np.array([0, 0, 1, 1, 2], np.int32)
    f = T.refit_event(u, v, labels, 4, p, GEOM)
    assert float(f[0].slope) == 0.25 and float(f[0].intercept) == 4.5    # the line through two points
    assert f[1].flags & T.FIT_DEGENERATE and f[1].n_hits == 2            # both hits at u = 5: no slope (plane artefact, A21)
    assert f[2].flags & T.FIT_DEGENERATE and f[2].n_hits == 1
    assert f[3].n_hits == 0 and f[3].plane_mask == 0 and f[3].max_run == 0 and f[3].flags == T.FIT_DEGENERATE


def test_plane_index_is_the_nearest_plane():
    for u in np.arange(-100.0, 100.0, 0.015625 * 37):
        uq = round(u * 64)
        want = math.floor((uq / 64 + 94.0) / 4.0 + 0.5)
        assert T.plane_index(uq, GEOM, 6) == want


def test_longest_run_brute_force():
    rng = np.random.default_rng(12)
    for _ in range(300):
        n = int(rng.integers(1, 65))
        mask = int(rng.integers(0, 2 ** 62)) & (2 ** n - 1)
        s = "".join("1" if (mask >> i) & 1 else "0" for i in range(n))
        assert T.longest_run(mask, n, False) == max((len(x) for x in s.split("0")), default=0)
        cyc = max((len(x) for x in (s + s).split("0")), default=0)
        assert T.longest_run(mask, n, True) == min(cyc, n)
    assert T.longest_run(0b1111100000, 10, False) == 5 and T.longest_run(0b1100000111, 10, True) == 5   # five in a row


def test_found_criterion_on_a_track_with_gaps():
    p = std_params(256, 256)
    uu, vv = synth.ideal_track(0.5, 3.0)
    keep = np.ones(48, bool); keep[[4, 9, 14, 19, 24, 29, 34, 39, 44]] = False      # every fifth plane missing: runs of 4
    f = T.refit_event(uu[keep], vv[keep], np.zeros(int(keep.sum()), np.int32), 1, p, GEOM)[0]
    assert f.max_run == 4 and not (f.flags & T.FIT_FOUND)
    keep[4] = True
    f = T.refit_event(uu[keep], vv[keep], np.zeros(int(keep.sum()), np.int32), 1, p, GEOM)[0]
    assert f.max_run == 9 and (f.flags & T.FIT_FOUND)


# ----------------------------------------------------------------------------- O13 peel-off
def test_peel_off_finds_ideal_tracks_one_by_one():
    p = std_params(64, 128, T=20, K=8, w_bins=1.5)
    us, vs = [], []
    for m, c in ((0.5, 20.0), (-0.25, -60.0), (0.0, 90.0)):
        uu, vv = synth.ideal_track(m, c)
        us.append(uu); vs.append(vv)
    rng = np.random.default_rng(13)
    us.append(rng.uniform(-94, 94, 10).astype(np.float32)); vs.append(rng.uniform(-194, 194, 10).astype(np.float32))
    u, v = np.concatenate(us), np.concatenate(vs)
    tracks, labels = T.peel_event(u, v, p)
    assert len(tracks) == 3
    assert tracks[0][2] >= tracks[1][2] >= tracks[2][2] >= 20               # remaining maxima can only shrink
    for s in range(3):
        got = set(np.nonzero(labels == s)[0])
        truth = [set(range(48 * j, 48 * j + 48)) for j in range(3)]
        assert max(len(got & tr) for tr in truth) >= 40                     # each peeled track is one of the true lines
    # the first track equals the best candidate of the one-pass search (same total order)
    acc = D.vote_event(u, v, p)
    cands, _ = D.find_clusters_event(acc, p)
    assert (tracks[0][0], tracks[0][1], tracks[0][2]) == (cands[0].theta_bin, cands[0].rho_bin, cands[0].votes)


# ----------------------------------------------------------------------------- O14 two-stage (coarse -> fine) Hough
def test_two_stage_with_unit_factors_reproduces_patch_maxima_of_the_exact_histogram():
    """c_theta = c_rho = 1: the coarse histogram IS the exact one, so every exact peak is a coarse peak and the maximum of its
    3 x 3 patch is the peak itself: the two-stage list equals the one-pass list (O4, O6) without the cluster fields."""
    p = std_params(64, 64, T=10, K=16)
    u, v = peel_case_like(21)
    two, n2 = T.two_stage_event(u, v, p, 1, 1)
    acc = D.vote_event(u, v, p)
    cands, n1 = D.find_clusters_event(acc, p)
    assert n1 <= p.max_candidates
    assert two == [(c.theta_bin, c.rho_bin, c.votes) for c in cands] and n2 == n1


def test_two_stage_candidates_carry_exact_counts_and_find_the_tracks():
    p = std_params(180, 256, T=24, K=16)
    u, v = peel_case_like(22, n_tracks=3, n_noise=15)
    acc = D.vote_event(u, v, p)
    for ct, cr in ((4, 4), (3, 8), (6, 2)):
        two, n2 = T.two_stage_event(u, v, p, ct, cr)
        assert n2 == len(two) >= 2                                           # (close tracks can share one coarse peak)
        for t, r, c in two:
            assert acc[t, r] == c                                            # fine patches are filled exactly as O3 does
        assert two == sorted(two, key=lambda x: (-x[2], x[0] * p.n_rho + x[1]))
        # (the method is an approximation: a track whose coarse bin is not a coarse local maximum is missed -- the exact global
        # maximum of this event, 36 votes, is not in the 4 x 4 list.  That is the paper's design, reading B8, not a defect.)
        assert all(c >= p.vote_threshold for _, _, c in two)


def peel_case_like(seed, n_tracks=2, n_noise=8):
    rng = np.random.default_rng(seed)
    us, vs = [], []
    for _ in range(n_tracks):
        uu, vv = synth.ideal_track(rng.uniform(-1, 1), rng.uniform(-100, 100))
        us.append(uu); vs.append(vv + rng.normal(0, 0.1, 48).astype(np.float32))
    us.append(rng.uniform(-94, 94, n_noise).astype(np.float32)); vs.append(rng.uniform(-194, 194, n_noise).astype(np.float32))
    return np.concatenate(us), np.concatenate(vs)
