"""Pins of the CPU oracle (both twins: pure-Python definition oracle and plain C oracle) against what the paper
and the mathematics fix: worked values, closed forms, invariants, library special cases, brute force.
No GPU, no product code: only oracle/ and the input generator are imported.

Pin numbering follows DESIGN.md "Pins" (P1 ... P14)."""
import itertools
import math
import zlib

import numpy as np
import pytest

from oracle import hough_c as C
from oracle import hough_def as D
from paper_2511_02742_b200 import synth
from util import cands_as_tuples, params_of, read_golden_table, std_params


# ----------------------------------------------------------------------------- two oracle front ends
class DefImpl:
    name = "def"

    @staticmethod
    def vote(u, v, p):
        return D.vote_event(u, v, p)

    @staticmethod
    def clusters(acc, p):
        return D.find_clusters_event(np.asarray(acc), p)

    @staticmethod
    def assign(u, v, cands, p):
        return D.assign_event(u, v, cands, p)

    @staticmethod
    def digest(acc):
        return D.digest(np.asarray(acc))

    @staticmethod
    def constants(p):
        k = D.constants(p)
        return k.H, k.F, k.Oq, k.Wq, np.array(k.Cq, np.int64), np.array(k.Sq, np.int64)


class CImpl:
    name = "c"
    vote = staticmethod(C.vote_event)
    clusters = staticmethod(C.find_clusters_event)
    assign = staticmethod(C.assign_event)
    digest = staticmethod(C.digest)
    constants = staticmethod(C.constants)


IMPLS = [DefImpl, CImpl]


@pytest.fixture(params=IMPLS, ids=lambda i: i.name)
def impl(request):
    return request.param


def run(impl, u, v, p):
    acc = impl.vote(u, v, p)
    cands, nf = impl.clusters(acc, p)
    labels = impl.assign(u, v, cands, p)
    return np.asarray(acc), cands, nf, np.asarray(labels)


def small_event(seed, n_tracks=2, n_noise=12):
    rng = np.random.default_rng(seed)
    us, vs = [], []
    for _ in range(n_tracks):
        m, c = rng.uniform(-1, 1), rng.uniform(-100, 100)
        uu, vv = synth.ideal_track(m, c)
        us.append(uu)
        vs.append(vv + rng.normal(0, 0.1, 48).astype(np.float32))
    us.append(rng.uniform(-94, 94, n_noise).astype(np.float32))
    vs.append(rng.uniform(-194, 194, n_noise).astype(np.float32))
    u, v = np.concatenate(us), np.concatenate(vs)
    perm = rng.permutation(len(u))
    return u[perm], v[perm]


# ----------------------------------------------------------------------------- P1 worked values
def test_p1_worked_values(impl):
    p = std_params(256, 256)
    H, F, Oq, Wq, Cq, Sq = impl.constants(p)
    assert (H, F, Oq) == (6, 22, 536870912)
    assert Wq == 2 ** 22                       # w = 1 bin = d_rho  ->  2^F
    rows = read_golden_table("p1_worked_values.txt")
    assert len(rows) == 6
    acc = np.asarray(impl.vote(np.array([10.0], np.float32), np.array([20.0], np.float32), p))
    for t, c, s, a, r in [[int(x) for x in row] for row in rows]:
        assert Cq[t] == c and Sq[t] == s
        assert 640 * int(Cq[t]) + 1280 * int(Sq[t]) + Oq == a
        assert a >> F == r
        assert acc[t, r] == 1 and acc[t].sum() == 1


def test_p1_frac_bits_of_all_config_grids(impl):
    # F = 23/22/21/20 for n_rho = 128/256/512/1024 on rho in [-256,256), coord_max 256
    for n_rho, F_exp in ((128, 23), (256, 22), (512, 21), (1024, 20)):
        H, F, Oq, _, Cq, Sq = impl.constants(std_params(64, n_rho))
        assert F == F_exp and Oq == 2 ** 29 and Cq[0] == 32768 and Sq[32] == 32768


# ----------------------------------------------------------------------------- P1b rounding rules (reading A5)
def _quantised(impl, x):
    """u_q and v_q of the hit (x, -x) as the oracle computes them, read off the two axis rows of a grid with d_rho = 2^-H:
    there C_q[0] = S_q[1] = 2^F exactly, so r = q + n_rho / 2 in both rows."""
    p = D.Params(2, 32, -16 / 64, 16 / 64, 0.2, 1, 1 / 64, 4, 6, -1)
    acc = np.asarray(impl.vote(np.array([x], np.float32), np.array([-x], np.float32), p))
    assert acc[0].sum() == 1 and acc[1].sum() == 1
    return int(np.argmax(acc[0])) - 16, int(np.argmax(acc[1])) - 16


def test_p1b_hit_rounding_is_ties_to_even(impl):
    rows = [r for r in read_golden_table("tie_rounding.txt") if r[0] == "hit"]
    assert len(rows) == 7
    for _, x, q in rows:
        x, q = float(x), int(q)
        assert float(np.float32(x)) == x and (x * 128) % 2 == 1            # an exact tie in fp32
        uq, vq = _quantised(impl, x)
        assert uq == q, (x, uq, q)
        assert vq == -q, (x, vq, q)                                          # rint is odd-symmetric
    # non-ties still round to nearest
    assert _quantised(impl, 0.0234375 + 2 ** -12)[0] == 2 and _quantised(impl, 0.0390625 + 2 ** -12)[0] == 3


def test_p1b_offset_and_window_round_half_away(impl):
    rows = [r for r in read_golden_table("tie_rounding.txt") if r[0] == "const"]
    assert len(rows) == 2
    for _, rho_min, w, oq, wq in rows:
        rho_min, w = float(rho_min), float(w)
        p = D.Params(8, 64, rho_min, rho_min + 64.0, 20.0, 3, w, 4, 6, 8)
        assert (p.rho_max - p.rho_min) / p.n_rho == 1.0
        H, F, Oq, Wq, _, _ = impl.constants(p)
        assert (H, F) == (6, 8)
        assert Oq == int(oq) and Wq == int(wq)


def test_p1b_default_frac_bits_keeps_the_bin_centres_in_int32(impl):
    """A rho range much wider than the hits (n_rho + 1 > the O3 span): F must shrink until (n_rho + 1) 2^F fits int32, so that the
    bin centres of O7 do.  1025 * 2^20 < 2^31 - 1 < 1025 * 2^21."""
    p = D.Params(16, 1024, -1.5, 1.5, 1.0, 2, 3.0 / 1024, 4, 6, -1)
    H, F, Oq, Wq, Cq, Sq = impl.constants(p)
    assert F == 20 and (p.n_rho + 1) * 2 ** F <= 2 ** 31 - 1 < (p.n_rho + 1) * 2 ** (F + 1)
    assert Oq == 512 * 2 ** 20 and Wq == 2 ** 20
    # the configs are unaffected (their O3 span exceeds n_rho + 1): F = 23 / 22 / 21 / 20 as before (test_p1_frac_bits...)


def test_p1c_theta_window(impl):
    """Restricted theta window: theta_t = theta_min + (theta_max - theta_min) t / n_theta.  Closed forms at
    the window's start, agreement with the rows of the full grid that sample the same angles, and the ideal-track peak (P5)."""
    from dataclasses import replace
    full = std_params(512, 256)
    win = replace(std_params(256, 256), theta_min=math.pi / 4, theta_max=3 * math.pi / 4)
    H, F, Oq, Wq, Cf, Sf = impl.constants(full)
    Hw, Fw, Oqw, Wqw, Cw, Sw = impl.constants(win)
    assert (Hw, Fw, Oqw, Wqw) == (H, F, Oq, Wq)
    assert Cw[0] == Sw[0] == 23170 and Cw[128] == 0 and Sw[128] == 32768          # 45 degrees: M / sqrt(2); 90 degrees: (0, M)
    assert np.abs(Cw - Cf[128:384]).max() <= 1 and np.abs(Sw - Sf[128:384]).max() <= 1   # same angles, last-bit rounding of theta only
    assert (Cw == Cf[128:384]).mean() > 0.9
    quarter = replace(std_params(64, 256), theta_min=math.pi / 2, theta_max=math.pi)
    _, _, _, _, Cq, Sq = impl.constants(quarter)
    assert Cq[0] == 0 and Sq[0] == 32768 and Cq[32] == -23170                         # 90 and 135 degrees
    # P5 in the window: a noiseless track through the centre of bin (t*, r*) of the windowed grid
    t_star, r_star = 70, 150
    th = math.pi / 4 + (math.pi / 2) * t_star / 256
    m, c = -1.0 / math.tan(th), (-256.0 + (r_star + 0.5) * 2.0) / math.sin(th)
    uu, vv = synth.ideal_track(m, c)
    acc = np.asarray(impl.vote(uu, vv, win))
    assert acc[t_star, r_star] == 48 == acc.max()
    cands, nf = impl.clusters(acc, win)
    c0 = cands[0]
    tb = c0.theta_bin if hasattr(c0, "theta_bin") else c0["theta_bin"]
    thf = c0.theta if hasattr(c0, "theta") else c0["theta"]
    assert acc[int(tb)].max() == 48 and abs(float(thf) - (math.pi / 4 + (math.pi / 2) * int(tb) / 256)) < 1e-6


def test_p1b_default_frac_bits_passes_the_int32_proof_on_exotic_plans():
    """d_rho far below the hit resolution 2^-H (found by tests/emu/fuzz_parity.py): the closed-form span is not enough there, F is
    lowered until q_max (|C_q| + |S_q|) + |O_q| fits for the corner hits; the corner hits then really do stay inside int32."""
    for p in (D.Params(180, 1000, -3.6, 2.4, 1.0, 1, 0.006, 16, 0, -1), D.Params(32, 568, -1.0, 1.0, 1.0, 5, 0.001, 16, 0, -1),
              D.Params(64, 700, -0.4, 0.4, 50.0, 2, 0.01, 8, 3, -1), D.Params(90, 300, -2.0, 3.0, 256.0, 2, 0.1, 8, 0, -1)):
        F = D.default_frac_bits(p)
        assert D.int32_proof(p, F) and (F == 24 or not D.int32_proof(p, F + 1) or
                                        (math.sqrt(2.0) * p.coord_max + max(abs(p.rho_min), abs(p.rho_max))) / ((p.rho_max - p.rho_min) / p.n_rho) * 2 ** (F + 1) > 2 ** 31 - 1)
        assert C.constants(p)[1] == F
        c = np.float32(p.coord_max)
        acc = D.vote_event(np.array([c, -c, c, -c], np.float32), np.array([c, c, -c, -c], np.float32), p)      # asserts the bound inside
        np.testing.assert_array_equal(acc, C.vote_event(np.array([c, -c, c, -c], np.float32), np.array([c, c, -c, -c], np.float32), p))


# ----------------------------------------------------------------------------- P2 table CRC
def test_p2_table_crc32(impl):
    for n_theta, crc in read_golden_table("table_crc32.txt"):
        n_theta = int(n_theta)
        n_rho = {180: 256, 256: 256, 512: 512, 128: 128, 1024: 1024}[n_theta]
        _, _, _, _, Cq, Sq = impl.constants(std_params(n_theta, n_rho))
        blob = np.concatenate([Cq, Sq]).astype("<i4").tobytes()
        assert f"{zlib.crc32(blob) & 0xffffffff:08x}" == crc


def test_p2_table_symmetries(impl):
    # cos(pi - x) = -cos x, sin(pi - x) = sin x, cos(pi/2 - x) = sin x: the rounded tables inherit them (up to libm ulps)
    _, _, _, _, Cq, Sq = impl.constants(std_params(512, 512))
    n = 512
    assert Cq[0] == 32768 and Sq[0] == 0 and Cq[n // 2] == 0 and Sq[n // 2] == 32768
    for t in range(1, n):
        assert abs(int(Cq[t]) + int(Cq[n - t])) <= 1 and abs(int(Sq[t]) - int(Sq[n - t])) <= 1
    for t in range(0, n // 2 + 1):
        assert abs(int(Cq[t]) - int(Sq[n // 2 - t])) <= 1
        assert abs(int(Cq[t]) ** 2 + int(Sq[t]) ** 2 - 32768 ** 2) <= 2 * 32768     # |(C,S)| = M within rounding


# ----------------------------------------------------------------------------- P3 axis rows are plain 1-D histograms
@pytest.mark.parametrize("n_rho", [128, 256, 512])
def test_p3_axis_rows_equal_numpy_histogram(impl, n_rho):
    u, v = small_event(3, n_tracks=3, n_noise=40)
    p = std_params(64, n_rho)
    acc = np.asarray(impl.vote(u, v, p))
    uq = np.rint(u.astype(np.float64) * 64) / 64
    vq = np.rint(v.astype(np.float64) * 64) / 64
    # theta = 0: rho = u;  theta = pi/2: rho = v.  d_rho is a power of two, so the float histogram is exact.
    hu, _ = np.histogram(uq, bins=n_rho, range=(-256.0, 256.0))
    hv, _ = np.histogram(vq, bins=n_rho, range=(-256.0, 256.0))
    # numpy closes the last bin on the right; no hit sits at +256 here
    assert (acc[0] == hu).all()
    assert (acc[32] == hv).all()


# ----------------------------------------------------------------------------- P4 conservation
def test_p4_conservation(impl):
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 3)
    p = params_of(wl)
    for e in range(3):
        u, v = b.event(e)
        acc = np.asarray(impl.vote(u, v, p))
        # generator data: |rho| <= sqrt(94^2 + 194^2) < 256, every (hit, theta) pair is in range
        assert (acc.sum(axis=1) == len(u)).all()
        assert acc.sum() == len(u) * p.n_theta


def test_p4_out_of_range_votes_are_dropped(impl):
    # rho range narrower than the hits: count the in-range pairs in float64 away from edges
    p = D.Params(64, 100, -50.0, 50.0, 256.0, 2, 1.0, 16)
    rng = np.random.default_rng(5)
    u = rng.uniform(-200, 200, 60).astype(np.float32)
    v = rng.uniform(-200, 200, 60).astype(np.float32)
    acc = np.asarray(impl.vote(u, v, p))
    th = np.pi * np.arange(64) / 64
    rho = u[:, None].astype(np.float64) * np.cos(th) + v[:, None].astype(np.float64) * np.sin(th)
    inside = ((rho >= -50) & (rho < 50)).sum()
    near_edge = ((np.abs(rho + 50) < 0.05) | (np.abs(rho - 50) < 0.05)).sum()
    assert abs(int(acc.sum()) - int(inside)) <= near_edge
    assert 0 < acc.sum() < 60 * 64


# ----------------------------------------------------------------------------- P5 single ideal track
@pytest.mark.parametrize("grid,t_star,r_star", [((256, 256), 90, 150), ((512, 512), 200, 300), ((180, 256), 60, 100),
                                                ((1024, 1024), 600, 411)])
def test_p5_single_ideal_track_peaks_at_its_analytic_bin(impl, grid, t_star, r_star):
    n_theta, n_rho = grid
    p = std_params(n_theta, n_rho, T=24)
    d_rho = 512.0 / n_rho
    th = math.pi * t_star / n_theta
    rho = -256.0 + (r_star + 0.5) * d_rho                # bin centre
    m, c = -1.0 / math.tan(th), rho / math.sin(th)        # v = m u + c  <=>  u cos(th) + v sin(th) = rho
    assert abs(m) <= 1.0
    u, v = synth.ideal_track(m, c)
    acc, cands, nf, labels = run(impl, u, v, p)
    assert acc[t_star, r_star] == 48 == acc.max()
    tup = cands_as_tuples(cands)
    assert nf >= 1 and (tup[0][0], tup[0][1], tup[0][2]) == (t_star, r_star, 48)
    assert (labels == 0).all()                            # every hit is within the window of its own line
    # fp32 parameters of the record: bin-centre rho and left-edge theta, 1e-5 relative (north_star)
    c0 = cands[0]
    th_rec = float(c0.theta if hasattr(c0, "theta") else c0["theta"])
    rho_rec = float(c0.rho if hasattr(c0, "rho") else c0["rho"])
    assert abs(th_rec - th) <= 1e-5 * abs(th) and abs(rho_rec - rho) <= 1e-5 * abs(rho)


# ----------------------------------------------------------------------------- P6 float cross-check
def test_p6_bins_agree_with_float64_evaluation(impl):
    u, v = small_event(11, n_tracks=3, n_noise=60)
    for n_theta, n_rho in ((256, 256), (512, 512), (256, 1024)):
        p = std_params(n_theta, n_rho)
        d_rho = 512.0 / n_rho
        acc = np.asarray(impl.vote(u, v, p))
        th = np.pi * np.arange(n_theta) / n_theta
        x = (u[:, None].astype(np.float64) * np.cos(th) + v[:, None].astype(np.float64) * np.sin(th) + 256.0) / d_rho
        rf = np.floor(x).astype(np.int64)
        ref = np.zeros_like(acc)
        np.add.at(ref, (np.broadcast_to(np.arange(n_theta), rf.shape), rf), 1)
        # the fixed-point result may move a vote by one bin only when the float rho is within 1/32 bin of an edge
        frac = x - np.floor(x)
        movable = int(((frac < 1 / 32) | (frac > 1 - 1 / 32)).sum())
        diff = np.abs(acc.astype(np.int64) - ref).sum()
        assert diff <= 2 * movable
        assert diff < 0.02 * acc.sum()
        # and never by more than one bin: row-wise cumulative sums differ by at most the movable count
        assert np.abs(np.cumsum(acc - ref, axis=1)).max() <= 3


# ----------------------------------------------------------------------------- P7 permutation invariance
def test_p7_permutation_invariance(impl):
    u, v = small_event(21, n_tracks=3, n_noise=30)
    p = std_params(180, 256, T=20)
    acc, cands, nf, labels = run(impl, u, v, p)
    perm = np.random.default_rng(0).permutation(len(u))
    acc2, cands2, nf2, labels2 = run(impl, u[perm], v[perm], p)
    assert (acc == acc2).all() and nf == nf2 and cands_as_tuples(cands) == cands_as_tuples(cands2)
    assert (labels[perm] == labels2).all()


# ----------------------------------------------------------------------------- P8 superposition
def test_p8_superposition(impl):
    from hypothesis import given, settings, strategies as st

    p = std_params(32, 64, T=2)
    coord = st.floats(min_value=-256.0, max_value=256.0, allow_nan=False, width=32)
    hits = st.lists(st.tuples(coord, coord), min_size=0, max_size=12)

    @settings(max_examples=25 if impl is DefImpl else 100, deadline=None)
    @given(hits, hits)
    def prop(a, b):
        ua, va = np.array([h[0] for h in a], np.float32), np.array([h[1] for h in a], np.float32)
        ub, vb = np.array([h[0] for h in b], np.float32), np.array([h[1] for h in b], np.float32)
        acc_ab = np.asarray(impl.vote(np.concatenate([ua, ub]), np.concatenate([va, vb]), p))
        assert (acc_ab == np.asarray(impl.vote(ua, va, p)) + np.asarray(impl.vote(ub, vb, p))).all()
        assert acc_ab.sum() <= (len(a) + len(b)) * p.n_theta

    prop()


# ----------------------------------------------------------------------------- P9 CCL against scipy.ndimage.label
def _random_acc(rng, n_theta, n_rho, T, density):
    acc = rng.integers(0, T, size=(n_theta, n_rho))
    on = rng.random((n_theta, n_rho)) < density
    acc[on] = rng.integers(T, T + 4, size=int(on.sum()))      # few distinct values -> many ties / plateaus
    return acc.astype(np.int32)


@pytest.mark.parametrize("density", [0.02, 0.15, 0.45, 0.9])
def test_p9_components_equal_scipy_label(impl, density):
    from scipy import ndimage

    rng = np.random.default_rng(int(density * 100))
    n_theta, n_rho, T = 24, 40, 5
    acc = _random_acc(rng, n_theta, n_rho, T, density)
    p = D.Params(n_theta, n_rho, -1.0, 1.0, 1.0, T, 0.1, n_theta * n_rho)     # K large: nothing truncated
    cands, nf = impl.clusters(acc, p)
    tup = cands_as_tuples(cands)
    assert nf == len(tup)
    lab, n_comp = ndimage.label(acc >= T, structure=np.ones((3, 3), int))
    sizes = ndimage.sum_labels(np.ones_like(acc), lab, index=np.arange(1, n_comp + 1)).astype(int)
    # every component has exactly one root record (cluster_root == own slot), and its size matches scipy's
    roots = [s for s, c in enumerate(tup) if c[3] == s]
    assert len(roots) == n_comp
    assert sum(tup[s][4] for s in roots) == int((acc >= T).sum())
    for s, (t, r, votes, root, nb) in enumerate(tup):
        cid = lab[t, r]
        assert cid > 0 and nb == sizes[cid - 1]
        rt, rr = tup[root][0], tup[root][1]
        assert lab[rt, rr] == cid                                  # root lies in the same scipy component
        in_comp = lab == cid
        best = max(((int(acc[a, b]), -(a * n_rho + b)) for a, b in zip(*np.nonzero(in_comp))))
        assert (tup[root][2], -(rt * n_rho + rr)) == best          # and is its max-key bin


def test_p9_peaks_are_the_strict_local_maxima_brute_force(impl):
    rng = np.random.default_rng(77)
    n_theta, n_rho, T = 17, 23, 4
    acc = _random_acc(rng, n_theta, n_rho, T, 0.3)
    p = D.Params(n_theta, n_rho, -1.0, 1.0, 1.0, T, 0.1, n_theta * n_rho)
    cands, nf = impl.clusters(acc, p)
    got = {(t, r) for t, r, *_ in cands_as_tuples(cands)}
    pad = np.full((n_theta + 2, n_rho + 2), -1, np.int64)
    pad[1:-1, 1:-1] = acc
    exp = set()
    for t in range(n_theta):
        for r in range(n_rho):
            if acc[t, r] < T:
                continue
            ok = True
            for dt, dr in itertools.product((-1, 0, 1), repeat=2):
                if (dt, dr) == (0, 0):
                    continue
                nv = pad[t + 1 + dt, r + 1 + dr]
                # neighbour wins on a larger count, or an equal count and a smaller linear index
                if nv > acc[t, r] or (nv == acc[t, r] and (dt < 0 or (dt == 0 and dr < 0))):
                    ok = False
            if ok:
                exp.add((t, r))
    assert got == exp and nf == len(exp)


# ----------------------------------------------------------------------------- P9w theta wrap (reading B9)
def _stack_of_copies(acc, k):
    """The accumulator continued over theta in [-k pi, (k + 1) pi): copy j is the grid itself for even j and the grid with its
    rho bins reversed for odd j (the line (theta + pi, rho) is the line (theta, -rho)).  -> (stack, row of copy 0's row 0)"""
    copies = [acc if j % 2 == 0 else acc[:, ::-1] for j in range(-k, k + 1)]
    return np.concatenate(copies, axis=0), k * acc.shape[0]


def _wrap_params(n_theta, n_rho, T, K=None):
    return D.Params(n_theta, n_rho, -1.0, 1.0, 1.0, T, 0.1, K or n_theta * n_rho, theta_wrap=True)


@pytest.mark.parametrize("shape,density,seed", [((5, 6), 0.5, 1), ((7, 9), 0.35, 2), ((3, 8), 0.6, 3), ((12, 10), 0.2, 4),
                                                 ((6, 7), 0.95, 5), ((9, 4), 0.05, 6)])
def test_p9w_wrap_equals_plain_rules_on_the_unrolled_theta_axis(impl, shape, density, seed):
    """Brute force: unroll the theta axis (stack mirrored copies), apply the NO-wrap definitions there with library labelling,
    and read the result off copy 0.  A simple path visits each bin at most once and moves at most one row per step, so
    n_rho + 1 copies on either side hold a lift of every path that starts in copy 0."""
    from scipy import ndimage

    rng = np.random.default_rng(seed)
    n_theta, n_rho, T = shape[0], shape[1], 3
    acc = _random_acc(rng, n_theta, n_rho, T, density)
    p = _wrap_params(n_theta, n_rho, T)
    cands, nf = impl.clusters(acc, p)
    tup = cands_as_tuples(cands)
    k = n_rho + 1
    stack, row0 = _stack_of_copies(acc, k)
    lin = np.arange(n_theta * n_rho).reshape(n_theta, n_rho)                 # linear index of the bin a stack cell is a copy of
    lin_stack, _ = _stack_of_copies(lin, k)
    # peaks: strict local maxima of copy 0 inside the stack under (count, -linear index of the original bin)
    exp_peaks = set()
    for t in range(n_theta):
        for r in range(n_rho):
            if acc[t, r] < T:
                continue
            me = (int(acc[t, r]), -int(lin[t, r]))
            ok = True
            for dt, dr in itertools.product((-1, 0, 1), repeat=2):
                tt, rr = row0 + t + dt, r + dr
                if (dt, dr) != (0, 0) and 0 <= rr < n_rho and (int(stack[tt, rr]), -int(lin_stack[tt, rr])) > me:
                    ok = False
            if ok:
                exp_peaks.add((t, r))
    assert {(t, r) for t, r, *_ in tup} == exp_peaks and nf == len(exp_peaks)
    # components: two bins belong together iff copy 0 of one is connected to SOME copy of the other
    lab, _ = ndimage.label(stack >= T, structure=np.ones((3, 3), int))
    classes = {}                                                             # stack label -> set of original bins
    for (tt, rr), l in np.ndenumerate(lab):
        if l:
            classes.setdefault(l, set()).add(int(lin_stack[tt, rr]))
    for s, (t, r, votes, root, nb) in enumerate(tup):
        members = classes[lab[row0 + t, r]]
        assert nb == len(members), (s, t, r)
        rt, rr = tup[root][0], tup[root][1]
        assert rt * n_rho + rr in members
        assert (tup[root][2], -(rt * n_rho + rr)) == max((int(acc.flat[b]), -b) for b in members)


def test_p9w_hand_built_seam_cases(impl):
    """Special cases small enough to check by eye: two on bins, one in the first and one in the last theta row."""
    n_theta, n_rho, T = 6, 10, 5
    plain, wrap = D.Params(n_theta, n_rho, -1.0, 1.0, 1.0, T, 0.1, 8), _wrap_params(n_theta, n_rho, T, 8)

    def both(cells):
        acc = np.zeros((n_theta, n_rho), np.int32)
        for (t, r), c in cells.items():
            acc[t, r] = c
        return cands_as_tuples(impl.clusters(acc, plain)[0]), cands_as_tuples(impl.clusters(acc, wrap)[0])

    r = 3
    m = n_rho - 1 - r                                                        # the bin that (0, r) continues into past the seam
    for dm in (-1, 0, 1):                                                    # straight and diagonal neighbours across the seam
        pl, wr = both({(0, r): 10, (n_theta - 1, m + dm): 9})
        assert pl == [(0, r, 10, 0, 1), (n_theta - 1, m + dm, 9, 1, 1)]
        assert wr == [(0, r, 10, 0, 2)]
        pl, wr = both({(0, r): 9, (n_theta - 1, m + dm): 10})
        assert wr == [(n_theta - 1, m + dm, 10, 0, 2)]
        pl, wr = both({(0, r): 10, (n_theta - 1, m + dm): 10})               # a tie: the smaller linear index wins
        assert wr == [(0, r, 10, 0, 2)]
    for dm in (-2, 2):                                                       # two bins apart: not neighbours
        pl, wr = both({(0, r): 10, (n_theta - 1, m + dm): 9})
        assert wr == pl == [(0, r, 10, 0, 1), (n_theta - 1, m + dm, 9, 1, 1)]
    pl, wr = both({(0, r): 10, (n_theta - 1, r): 9})                         # same rho bin, NOT mirrored: r = 3 continues into 6, not 3
    assert wr == pl and len(wr) == 2
    pl, wr = both({(0, 0): 10, (n_theta - 1, n_rho - 1): 9, (0, n_rho - 1): 8, (n_theta - 1, 0): 7})   # the corners pair up crosswise
    assert wr == [(0, 0, 10, 0, 2), (0, n_rho - 1, 8, 1, 2)]


def test_p9w_a_vertical_track_is_one_cluster_with_wrap_and_two_without(impl):
    """Textbook case: hits on the line u = c (theta = 0) vote (0, bin(c)) n times, and the rows just below theta = pi see the
    same line at rho = -c: the ridge of a single track crosses the seam.  Without wrap it is two clusters, each with its own
    best candidate; with wrap (B9) one cluster whose size is the sum, rooted at the better of the two."""
    n_theta, n_rho = 90, 64
    c = -256.0 + 45.5 * (512.0 / n_rho)                                      # centre of rho bin 45
    v = np.linspace(-30, 30, 25).astype(np.float32)
    u = np.full_like(v, c)
    base = dict(n_theta=n_theta, n_rho=n_rho, rho_min=-256.0, rho_max=256.0, coord_max=256.0, vote_threshold=12,
                assign_window=8.0, max_candidates=16)
    acc = impl.vote(u, v, D.Params(**base))
    assert acc[0, 45] == len(u) and acc[n_theta - 1, n_rho - 1 - 45] >= 12   # both sides of the seam are on
    plain = cands_as_tuples(impl.clusters(acc, D.Params(**base))[0])
    wrapped = cands_as_tuples(impl.clusters(acc, D.Params(**base, theta_wrap=True))[0])
    assert {(t, r) for t, r, *_ in wrapped} <= {(t, r) for t, r, *_ in plain}    # more neighbours can only remove peaks
    roots_plain = sorted({rt for *_, rt, _ in plain})
    assert len(roots_plain) == 2 and plain[0][:2] == (0, 45)
    near, far = (plain[rt] for rt in roots_plain)
    assert near[0] < 10 and far[0] > n_theta - 10                            # one cluster on either side of the seam
    assert {rt for *_, rt, _ in wrapped} == {0} and wrapped[0][:3] == (0, 45, len(u))
    assert all(nb == near[4] + far[4] for *_, nb in wrapped)


def test_p9w_rotating_the_theta_origin_changes_nothing(impl):
    """Invariant: with wrap the theta axis has no preferred origin.  Rotating the rows by s (rows pushed past the seam come
    back mirrored) maps peaks to peaks and clusters to clusters when no two bins tie (all counts distinct)."""
    rng = np.random.default_rng(9)
    n_theta, n_rho, T = 8, 11, 40
    acc = rng.permutation(n_theta * n_rho).reshape(n_theta, n_rho).astype(np.int32)
    p = _wrap_params(n_theta, n_rho, T)
    ref = cands_as_tuples(impl.clusters(acc, p)[0])
    for s in (1, 3, 7):
        rot = np.concatenate([acc[s:], acc[:s, ::-1]], axis=0)
        back = lambda t, r: (t + s, r) if t + s < n_theta else (t + s - n_theta, n_rho - 1 - r)
        got = cands_as_tuples(impl.clusters(rot, p)[0])
        assert sorted((back(t, r), vt, nb) for t, r, vt, _, nb in got) == sorted(((t, r), vt, nb) for t, r, vt, _, nb in ref)
        assert sorted(back(*got[rt][:2]) for *_, rt, _ in got) == sorted(ref[rt][:2] for *_, rt, _ in ref)


def test_p9w_wrap_needs_the_paper_window_and_a_symmetric_rho_range():
    acc = np.zeros((6, 6), np.int32)
    for bad in (D.Params(6, 6, -1.0, 2.0, 1.0, 1, 0.1, 4, theta_wrap=True), D.Params(2, 6, -1.0, 1.0, 1.0, 1, 0.1, 4, theta_wrap=True),
                D.Params(6, 6, -1.0, 1.0, 1.0, 1, 0.1, 4, theta_min=0.0, theta_max=1.0, theta_wrap=True)):
        with pytest.raises(AssertionError):
            D.find_clusters_event(acc, bad)
        with pytest.raises(RuntimeError):
            C.find_clusters_event(acc, bad)


def test_p9w_both_oracles_agree_with_wrap_on_generated_events():
    for seed in (1, 2, 3):
        u, v = small_event(seed, n_tracks=3, n_noise=30)
        u[:10] = np.float32(-93.5)                                           # a vertical track: its ridge crosses the seam
        p = std_params(64, 64, T=8, K=32, theta_wrap=True)
        a1, c1, n1, l1 = run(DefImpl, u, v, p)
        a2, c2, n2, l2 = run(CImpl, u, v, p)
        assert (a1 == a2).all() and n1 == n2 and cands_as_tuples(c1) == cands_as_tuples(c2) and (l1 == l2).all()
        assert [float(c.theta) for c in c1] == [float(c["theta"]) for c in c2]


# ----------------------------------------------------------------------------- P10 brute force over hit pairs
def _collinear_event(rng, p, groups, n_per_group, n_free):
    """Exactly collinear groups on bin-centre lines (well separated), plus general-position hits."""
    d_rho = (p.rho_max - p.rho_min) / p.n_rho
    lines = [(math.pi * t / p.n_theta, p.rho_min + (r + 0.5) * d_rho) for t, r in groups]

    def far_from_foreign_lines(uu, vv, own):
        return all(abs(uu * math.cos(th) + vv * math.sin(th) - rho) > 2 * d_rho
                   for g, (th, rho) in enumerate(lines) if g != own)

    us, vs, truth = [], [], []
    for g, (th, rho) in enumerate(lines):
        # points rho*(cos,sin) + s*(-sin,cos), s spread widely so neighbouring theta bins cannot collect them all;
        # a point near a crossing with another group's line would be ambiguous for the brute force: redraw it
        for s0 in np.linspace(-120, 120, n_per_group):
            spread = 3.0
            while True:
                s = s0 + rng.uniform(-spread, spread)
                spread *= 1.2
                uu = rho * math.cos(th) - s * math.sin(th)
                vv = rho * math.sin(th) + s * math.cos(th)
                if far_from_foreign_lines(uu, vv, g):
                    break
            us.append(uu)
            vs.append(vv)
            truth.append(g)
    for _ in range(n_free):
        while True:
            uu, vv = rng.uniform(-200, 200), rng.uniform(-200, 200)
            if far_from_foreign_lines(uu, vv, -1):
                break
        us.append(uu)
        vs.append(vv)
        truth.append(-1)
    return np.array(us, np.float32), np.array(vs, np.float32), np.array(truth)


@pytest.mark.parametrize("seed", [1, 2, 3, 4])
def test_p10_brute_force_line_through_hit_pairs(impl, seed):
    rng = np.random.default_rng(seed)
    T = 8
    p = std_params(128, 128, T=T, K=16, w_bins=0.25)         # window = the brute-force tolerance eps = d_rho / 4
    d_rho = 4.0
    groups = [(20 + 7 * seed, 40), (64, 75 + seed), (100 - 5 * seed, 60)]
    u, v, truth = _collinear_event(rng, p, groups, 10, 8)
    acc, cands, nf, labels = run(impl, u, v, p)
    # brute force: every hit pair defines a line; collect the hits within eps of it; keep the maximal sets with >= T hits
    eps = d_rho / 4
    ud, vd = u.astype(np.float64), v.astype(np.float64)
    sets = set()
    for i, j in itertools.combinations(range(len(u)), 2):
        dx, dy = ud[j] - ud[i], vd[j] - vd[i]
        n = math.hypot(dx, dy)
        if n < 1e-9:
            continue
        dist = np.abs((ud - ud[i]) * dy - (vd - vd[i]) * dx) / n
        members = frozenset(np.nonzero(dist <= eps)[0].tolist())
        if len(members) >= T:
            sets.add(members)
    maximal = [s for s in sets if not any(s < o for o in sets)]
    hough_sets = [frozenset(np.nonzero(labels == s)[0].tolist()) for s in range(min(nf, p.max_candidates))]
    assert nf == len(groups) == len(maximal)
    assert sorted(map(sorted, hough_sets)) == sorted(map(sorted, maximal))
    for s, hs in enumerate(hough_sets):                        # and each set is one generated group
        assert len(set(truth[list(hs)])) == 1 and truth[list(hs)][0] >= 0
    got_bins = sorted((t, r) for t, r, *_ in cands_as_tuples(cands))
    assert got_bins == sorted(groups)


# ----------------------------------------------------------------------------- P11 assignment invariants
def test_p11_assignment_invariants(impl):
    wl = synth.workload(2)
    b = synth.generate(wl, 0, 2)
    p = params_of(wl)
    H, F, Oq, Wq, Cq, Sq = impl.constants(p)
    for e in range(2):
        u, v = b.event(e)
        acc, cands, nf, labels = run(impl, u, v, p)
        tup = cands_as_tuples(cands)
        uq = np.rint(u.astype(np.float64) * 2 ** H).astype(np.int64)
        vq = np.rint(v.astype(np.float64) * 2 ** H).astype(np.int64)
        E = np.empty((len(u), len(tup)), np.int64)
        for s, (t, r, votes, _, _) in enumerate(tup):
            a = uq * int(Cq[t]) + vq * int(Sq[t]) + Oq
            E[:, s] = a - (r * 2 ** F + 2 ** (F - 1))
            # the votes of the peak bin are exactly the hits whose residual lies in the bin: -2^(F-1) <= e < 2^(F-1)
            assert votes == int(((E[:, s] >= -2 ** (F - 1)) & (E[:, s] < 2 ** (F - 1))).sum())
        absE = np.abs(E)
        for i in range(len(u)):
            elig = np.nonzero(absE[i] <= Wq)[0]
            if len(elig) == 0:
                assert labels[i] == -1
            else:
                best = elig[np.argmin(absE[i, elig])]             # argmin returns the first (lowest slot) minimum
                assert labels[i] == best
        assert (labels >= 0).mean() > 0.6                         # most hits of a 10-20 track event belong to a line


def test_p11_single_candidate_wide_window_labels_every_voter(impl):
    u, v = small_event(5, n_tracks=1, n_noise=20)
    p = std_params(256, 256, T=24, K=1, w_bins=0.5)              # W_q = 2^(F-1): window == the peak bin itself
    acc, cands, nf, labels = run(impl, u, v, p)
    (t, r, votes, _, _), = cands_as_tuples(cands)
    # hits labelled 0 are the voters of the peak bin plus, at most, hits exactly on its upper edge (|e| == 2^(F-1))
    assert votes <= int((labels == 0).sum()) <= votes + 1


# ----------------------------------------------------------------------------- P12 rank / root invariants
def test_p12_rank_and_root_invariants(impl):
    wl = synth.workload(3)
    b = synth.generate(wl, 0, 1)
    p = params_of(wl)
    u, v = b.event(0)
    acc = np.asarray(impl.vote(u, v, p))
    cands, nf = impl.clusters(acc, p)
    tup = cands_as_tuples(cands)
    assert nf > p.max_candidates == len(tup)                     # cfg3 is noise-saturated at T = 20: truncated to K
    keys = [(-c[2], c[0] * p.n_rho + c[1]) for c in tup]
    assert keys == sorted(keys)
    for s, c in enumerate(tup):
        assert 0 <= c[3] <= s and tup[c[3]][3] == c[3]            # root is kept, out-ranks its members, is its own root
        assert c[4] == tup[c[3]][4] and c[4] >= 1
        assert acc[c[0], c[1]] == c[2] >= p.vote_threshold
    # plane artefacts (reading A21): hits sharing a detector plane are collinear at theta = 0 -> 48 peaks in row 0
    row0 = [c for c in tup if c[0] == 0]
    assert len(row0) == 48
    # raising T never creates on-bins; n_found with a higher threshold counts a subset of the on-mask's maxima
    p_hi = params_of(wl, vote_threshold=30)
    _, nf_hi = impl.clusters(acc, p_hi)
    assert nf_hi <= nf and (acc >= 30).sum() <= (acc >= 20).sum()


# ----------------------------------------------------------------------------- P13 loose library cross-check
def test_p13_opencv_point_set_hough_agrees_within_a_bin(impl):
    cv2 = pytest.importorskip("cv2")
    u, v = small_event(9, n_tracks=1, n_noise=10)
    p = std_params(256, 256, T=24)
    acc, cands, nf, labels = run(impl, u, v, p)
    t0, r0 = cands_as_tuples(cands)[0][:2]
    pts = np.stack([u, v], axis=1).reshape(-1, 1, 2).astype(np.float32)
    d_rho, d_th = 2.0, math.pi / 256
    lines = cv2.HoughLinesPointSet(pts, 1, 24, -256.0, 256.0, d_rho, 0.0, math.pi - d_th / 2, d_th)
    votes, rho, theta = lines[0][0]
    assert abs(theta / d_th - t0) <= 1.01
    assert abs((rho + 256.0) / d_rho - (r0 + 0.5)) <= 1.51       # different rounding conventions: sanity only


# ----------------------------------------------------------------------------- P14 two oracles
def _same(a, b):
    return (np.asarray(a[0]) == np.asarray(b[0])).all() and cands_as_tuples(a[1]) == cands_as_tuples(b[1]) \
        and a[2] == b[2] and (a[3] == b[3]).all()


def test_p14_definition_oracle_equals_c_oracle_on_cfg0():
    wl = synth.workload(0)
    b = synth.generate(wl)
    p = params_of(wl)
    ra, rb = run(DefImpl, b.u, b.v, p), run(CImpl, b.u, b.v, p)
    assert _same(ra, rb)
    assert rb[2] == 3                                           # three tracks, three candidates
    fa = [(float(c.theta), float(c.rho)) for c in ra[1]]
    fb = [(float(c["theta"]), float(c["rho"])) for c in rb[1]]
    assert fa == fb
    assert DefImpl.digest(ra[0]) == CImpl.digest(rb[0])


def edge_cases():
    """(name, params, u, v): the adversarial set of DESIGN.md; hits only, usable by GPU parity tests too."""
    f32 = np.float32
    cases = []
    p = std_params(64, 64, T=3, K=8)
    cases.append(("empty", p, np.zeros(0, f32), np.zeros(0, f32)))
    cases.append(("all_invalid", p, np.array([np.nan, np.inf, -np.inf, 300.0, 1.0], f32),
                  np.array([1.0, 2.0, 3.0, 4.0, np.nan], f32)))
    cases.append(("coord_max_corners", p, np.array([256.0, -256.0, 256.0, -256.0, 256.00003], f32),
                  np.array([256.0, 256.0, -256.0, -256.0, 0.0], f32)))
    # hits whose fixed-point a is an exact multiple of 2^F in the axis rows (rho on a bin edge): u, v multiples of d_rho = 8
    g = np.arange(-248, 256, 8, dtype=f32)
    cases.append(("bin_edges", p, g, g[::-1].copy()))
    cases.append(("duplicates", p, np.full(500, 12.5, f32), np.full(500, -40.25, f32)))
    p1 = std_params(32, 32, T=1, K=4096)
    rng = np.random.default_rng(1)
    cases.append(("threshold_one_nfound_gt_K", std_params(32, 32, T=1, K=8), rng.uniform(-200, 200, 40).astype(f32),
                  rng.uniform(-200, 200, 40).astype(f32)))
    cases.append(("threshold_one_all_kept", p1, rng.uniform(-200, 200, 9).astype(f32), rng.uniform(-200, 200, 9).astype(f32)))
    # lines through grid borders / corners: theta = 0 row and last theta row, first and last rho bins
    ub = np.concatenate([np.full(6, -255.0, f32), np.full(6, 255.0, f32), np.linspace(-250, 250, 6).astype(f32)])
    vb = np.concatenate([np.linspace(-250, 250, 6).astype(f32), np.linspace(-250, 250, 6).astype(f32), np.full(6, 255.0, f32)])
    cases.append(("borders", std_params(64, 64, T=5, K=32), ub, vb))
    # the paper's own grid: 180 x 1000, rho in [-500, 500): d_rho = 1 but O_q not a power of two
    pp = D.Params(180, 1000, -500.0, 500.0, 360.0, 6, 1.0, 16)
    uu, vv = small_event(2, n_tracks=2, n_noise=10)
    cases.append(("paper_grid_180x1000", pp, uu, vv))
    # non-power-of-two d_rho and odd n_theta
    pn = D.Params(45, 77, -230.0, 245.0, 250.0, 6, 3.0, 16)
    cases.append(("odd_grid_nonpow2_drho", pn, uu, vv))
    # rounding ties (reading A5; goldens in tests/golden/tie_rounding.txt): hit coordinates at odd multiples of 2^-(H+1) on a
    # grid whose axis rows resolve single fixed-point steps, and offset / window constants with a fractional part of 1/2
    ties = np.array([0.0078125, 0.0234375, 0.0390625, 0.0546875, -0.0078125, -0.0234375, -0.0390625, 0.0234375, 0.0390625], f32)
    cases.append(("hit_rounding_ties", D.Params(2, 32, -16 / 64, 16 / 64, 0.2, 1, 1 / 64, 16, 6, -1), ties, -ties))
    for nm, rmin, w in (("llround_ties_pos_offset", -100.001953125, 1.001953125), ("llround_ties_neg_offset", 100.001953125, 2.501953125)):
        pc = D.Params(8, 64, rmin, rmin + 64.0, 20.0, 3, w, 4, 6, 8)
        sgn = -1.0 if rmin > 0 else 1.0
        cases.append((nm, pc, (sgn * np.linspace(-18, 18, 40)).astype(f32), np.linspace(-15, 19, 40).astype(f32)))
    # coordinates beyond 2^15 fixed-point units (coord_max 1000, H = 6): u_q^2 + v_q^2 exceeds 32 bits at the corners
    pw = D.Params(64, 512, -1415.0, 1415.0, 1000.0, 3, 6.0, 16, 6, -1)
    cw_u = np.concatenate([np.full(6, 1000.0, f32), np.full(6, -1000.0, f32), np.linspace(-990, 990, 12).astype(f32)])
    cw_v = np.concatenate([np.linspace(985, 1000, 6).astype(f32), np.linspace(-1000, -985, 6).astype(f32), np.linspace(-30, 30, 12).astype(f32)])
    cases.append(("wide_coordinates_corner_hits", pw, cw_u, cw_v))
    return cases


@pytest.mark.parametrize("case", edge_cases(), ids=lambda c: c[0])
def test_p14_edge_set_both_oracles_agree(case):
    name, p, u, v = case
    ra, rb = run(DefImpl, u, v, p), run(CImpl, u, v, p)
    assert _same(ra, rb)
    acc = ra[0]
    n_valid = int((np.isfinite(u) & np.isfinite(v) & (np.abs(u) <= p.coord_max) & (np.abs(v) <= p.coord_max)).sum())
    assert acc.sum() <= n_valid * p.n_theta
    assert (ra[3][~(np.isfinite(u) & np.isfinite(v))] == -1).all()
    if name in ("empty", "all_invalid"):
        assert acc.sum() == 0 and ra[2] == 0 and (ra[3] == -1).all()
    if name == "coord_max_corners":
        assert n_valid == 4 and acc[0].sum() == 2                 # u = +256 lands in bin n_rho (dropped), u = -256 in bin 0
    if name == "duplicates":
        assert acc.max() == 500 and (acc.sum(axis=1) == 500).all()
    if name == "threshold_one_nfound_gt_K":
        assert ra[2] > p.max_candidates == len(ra[1])


def test_p14_u16_boundary_65535_identical_hits():
    # one bin receives every hit: the largest count a 16-bit counter can hold (reading A16)
    p = std_params(8, 16, T=65535, K=4)
    u = np.full(65535, 3.0, np.float32)
    v = np.full(65535, 5.0, np.float32)
    acc = C.vote_event(u, v, p)
    assert acc.max() == 65535 and (acc.sum(axis=1) == 65535).all()
    cands, nf = C.find_clusters_event(acc, p)
    assert nf >= 1 and cands[0]["votes"] == 65535


# ----------------------------------------------------------------------------- O8 digest
def test_digest_is_splitmix64_weighted_sum(impl):
    # SplitMix64 reference outputs for seed 0 (Steele, Lea, Flood 2014; also the xoshiro seeding reference):
    assert D.mix64(0) == 0xE220A8397B1DCDAF
    assert D.mix64(0x9E3779B97F4A7C15) == 0x6E789E6AA1B965F4
    acc = np.zeros((4, 8), np.int32)
    assert impl.digest(acc) == 0
    acc[0, 0] = 1
    assert impl.digest(acc) == 0xE220A8397B1DCDAF
    acc[2, 5] = 3
    assert impl.digest(acc) == (0xE220A8397B1DCDAF + 3 * D.mix64(2 * 8 + 5)) % 2 ** 64
    rng = np.random.default_rng(3)
    a = rng.integers(0, 50, (6, 9)).astype(np.int32)
    b = rng.integers(0, 50, (6, 9)).astype(np.int32)
    assert impl.digest(a + b) == (impl.digest(a) + impl.digest(b)) % 2 ** 64       # linear


# ----------------------------------------------------------------------------- sanity: synthetic-truth efficiency
def test_synthetic_truth_efficiency_is_high():
    """PAPER.md Eq. 7.1 (L132-136) efficiency = N_found / N_all, on synthetic truth: a track counts as found if a
    candidate lies within +-1 bin of its analytic (theta*, rho*).  Sanity figure, not graded."""
    for cfg, n_ev in ((1, 20), (2, 5)):
        wl = synth.workload(cfg)
        b = synth.generate(wl, 0, n_ev)
        p = params_of(wl)
        res = C.run_batch(b.u, b.v, b.offsets, p, want_labels=False)
        found = total = 0
        for e in range(n_ev):
            nk = min(int(res["n_found"][e]), p.max_candidates)
            cb = {(int(c["theta_bin"]), int(c["rho_bin"])) for c in res["cands"][e][:nk]}
            for m, c in zip(b.track_m[b.track_offsets[e]:b.track_offsets[e + 1]], b.track_c[b.track_offsets[e]:b.track_offsets[e + 1]]):
                th = math.atan2(1.0, -m)
                t = th / math.pi * p.n_theta
                r = (c * math.sin(th) - p.rho_min) / wl.d_rho
                ts, rs = int(round(t)), int(math.floor(r))
                total += 1
                found += any((ts + dt, rs + dr) in cb for dt in (-1, 0, 1) for dr in (-1, 0, 1))
        assert found / total > 0.95
