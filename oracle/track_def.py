"""Definition oracle of the stages around the Hough core, in plain Python integers.

TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It shares no code with the CUDA path and never imports it.

  O9   refit        least-squares straight line through the hits assigned to a candidate     PAPER.md L94, L106 ("the
                    corresponding RecoHits lying along it are used as seeds"), L112-114 (seed fit; the helical fit itself
                    needs the detector geometry and is out of scope -- the straight line in the projection plane stands in)
  O10  found        "A track is regarded as found if its hits are reconstructed and clustered in continuous five vanes"
                                                                                             PAPER.md L136 (Sec. 7, Eq. 7.1)
  O11  slice        "the reconstructed hit points are divided into overlapping time windows of 10 ns, with a sliding step
                    of 5 ns"
  O12  phi          "(x, y, z) ... transformed into the (phi, z) space, where phi = atan(y / x)"
  O13  peel-off     "a peak-finding algorithm identifies the bin with the highest number of entries ... track seeds are found
                    by selecting the hits that align with the straight line" -- repeated on the remaining hits
                                                                                             PAPER.md L94, L106

Readings (B1-B8):
  B1  phi is measured in degrees, four-quadrant (atan2), in [-180, 180]; the paper's rho range -500...500 with z in +-200 mm
      only makes sense for phi in degrees.
  B2  phi is computed by integer CORDIC (vectoring mode) on fixed-point x, y with an angle table defined by formula, so that
      CPU and GPU agree bit for bit; it equals atan2 within the bound `cordic_error_bound_deg` (pinned against libm).
  B3  times are rounded to 2^-8 ns (ties to even); window w of a fill covers  t0 + w step <= t < t0 + w step + width.
  B4  within a window the hits keep their input order; invalid hits (non-finite, |x| or |y| above xy_max, x = y = 0) belong to
      no window.
  B5  the line refit is ordinary least squares v = slope u + intercept on the FIXED-POINT hit coordinates (the ones the vote
      uses), with exact integer sums and one rounding sequence in double; a candidate with fewer than two hits or with all
      hits at one u (a plane artefact, reading A21) has no slope: flag DEGENERATE, slope = intercept = 0.
  B6  plane (vane) index of a hit = nearest plane: floor((u - origin) / pitch + 1/2), counted only inside [0, n_planes);
      "continuous five" = a run of >= min_run consecutive plane indices that each hold >= 1 assigned hit; with wrap the
      planes form a ring (the 40 vanes of the detector).
  B8  two-stage (coarse -> fine) Hough, PAPER.md L124 / Fig. 5 ("a coarse-binning histogram followed by a fine-binning
      histogram"; no further detail in the paper): the coarse grid merges c_theta x c_rho fine bins; a coarse row T votes at
      the fine theta row in its middle, t_T = min(T c_theta + c_theta // 2, n_theta - 1), into coarse bin r_fine // c_rho;
      coarse peaks = strict local maxima >= T of the coarse histogram under the same total order, the best K kept; every kept
      coarse peak (T, R) opens a fine patch of the coarse bins T-1..T+1 x R-1..R+1 (clipped to the grid), filled exactly as
      O3 does; its candidate is the patch's maximum under (count, -L) if count >= T; duplicates are merged and the result is
      ranked like O6.  cluster_root = own slot, cluster_nbins = 0 (no clustering in this variant).
  B7  peel-off: the global maximum under the total order (count, -L); stop when its count < T or after K tracks; its hits are
      those within the assignment window of its bin-centre line; they are removed from the hit set and the histogram is
      refilled from the remaining hits (equivalently: their votes are subtracted); a maximum none of whose hits lies inside
      the window (window narrower than half a bin) ends the search.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

import numpy as np

from . import hough_def as D

FIT_DEGENERATE = 2
FIT_FOUND = 1


# ----------------------------------------------------------------------------- O9 / O10
@dataclass(frozen=True)
class PlaneGeometry:
    origin: float       # u of plane 0
    pitch: float        # distance between neighbouring planes (> 0)
    n_planes: int       # 1 ... 64
    min_run: int = 5
    wrap: bool = False  # planes form a ring


@dataclass(frozen=True)
class Fit:
    n_hits: int
    plane_mask: int
    max_run: int
    flags: int
    slope: np.float32
    intercept: np.float32


def plane_index(uq: int, g: PlaneGeometry, H: int) -> int:
    """B6: nearest plane of a fixed-point coordinate, floor((u - origin) / pitch + 1/2) in integers."""
    oq = D._llround(g.origin * float(2 ** H))
    pq = D._llround(g.pitch * float(2 ** H))
    assert pq >= 1
    return (2 * (uq - oq) + pq) // (2 * pq)


def longest_run(mask: int, n_planes: int, wrap: bool) -> int:
    """Longest run of consecutive set bits among bits 0 .. n_planes-1; cyclic if wrap."""
    bits = [(mask >> i) & 1 for i in range(n_planes)]
    if all(bits):
        return n_planes
    best = cur = 0
    seq = bits + bits if wrap else bits
    for b in seq:
        cur = cur + 1 if b else 0
        best = max(best, cur)
    return min(best, n_planes)


def refit_event(u: Sequence, v: Sequence, labels: Sequence[int], n_kept: int, p: D.Params, g: PlaneGeometry) -> List[Fit]:
    """O9 + O10 for one event: one Fit per kept candidate slot 0 .. n_kept-1."""
    k = D.constants(p)
    assert math.floor(p.coord_max * 2 ** k.H) <= 2 ** 15, "refit needs |u_q|, |v_q| <= 2^15 (exact 64-bit sums)"
    n = [0] * n_kept
    Su, Sv, Suu, Suv, mask = ([0] * n_kept for _ in range(5))
    for uu, vv, lab in zip(u, v, labels):
        if lab < 0:
            continue
        ok, uq, vq = D.quantise_hit(uu, vv, p, k)
        assert ok and lab < n_kept
        n[lab] += 1
        Su[lab] += uq; Sv[lab] += vq; Suu[lab] += uq * uq; Suv[lab] += uq * vq
        pl = plane_index(uq, g, k.H)
        if 0 <= pl < g.n_planes:
            mask[lab] |= 1 << pl
    out = []
    for s in range(n_kept):
        den = n[s] * Suu[s] - Su[s] * Su[s]
        num = n[s] * Suv[s] - Su[s] * Sv[s]
        assert abs(den) < 2 ** 63 and abs(num) < 2 ** 63
        run = longest_run(mask[s], g.n_planes, g.wrap)
        flags = FIT_FOUND if run >= g.min_run else 0
        if n[s] < 2 or den == 0:
            flags |= FIT_DEGENERATE
            slope = icpt = 0.0
        else:
            slope = float(num) / float(den)                                   # int64 -> double (round to nearest), one division
            icpt = (float(Sv[s]) - slope * float(Su[s])) / float(n[s])        # in fixed-point units
            icpt = icpt * (1.0 / float(2 ** k.H))                             # exact scaling back to hit units
        out.append(Fit(n[s], mask[s], run, flags, np.float32(slope), np.float32(icpt)))
    return out


# ----------------------------------------------------------------------------- O11 / O12
@dataclass(frozen=True)
class FrontEnd:
    t0: float = 0.0             # start of window 0 (ns)
    width: float = 10.0
    step: float = 5.0
    windows_per_fill: int = 8
    xy_max: float = 512.0       # |x|, |y| <= xy_max (mm)
    time_frac_bits: int = 8
    xy_frac_bits: int = 6
    phi_frac_bits: int = 16     # phi LSB = 2^-16 degree
    cordic_iterations: int = 20
    cordic_guard_bits: int = 14


def cordic_table(fe: FrontEnd) -> Tuple[int, ...]:
    """A_i = llround(atan(2^-i) * 180 / pi * 2^P), i = 0 .. N-1 (double precision, halves away from zero)."""
    return tuple(D._llround(math.atan(2.0 ** -i) * (180.0 / math.pi) * float(2 ** fe.phi_frac_bits)) for i in range(fe.cordic_iterations))


def cordic_phi_q(xq: int, yq: int, fe: FrontEnd) -> int:
    """B2: phi = atan2(y, x) in units of 2^-P degrees by integer CORDIC, vectoring mode.  (xq, yq) != (0, 0)."""
    assert (xq, yq) != (0, 0)
    A = cordic_table(fe)
    X, Y, Z = abs(xq) << fe.cordic_guard_bits, yq << fe.cordic_guard_bits, 0
    for i in range(fe.cordic_iterations):
        if Y >= 0:
            X, Y, Z = X + (Y >> i), Y - (X >> i), Z + A[i]        # >> floors (arithmetic shift)
        else:
            X, Y, Z = X - (Y >> i), Y + (X >> i), Z - A[i]
        assert abs(X) < 2 ** 31 and abs(Y) < 2 ** 31, "CORDIC state leaves int32"
    half_turn = 180 << fe.phi_frac_bits
    if xq >= 0:
        return Z
    return half_turn - Z if yq >= 0 else -half_turn - Z


def cordic_error_bound_deg(r_q: float, fe: FrontEnd) -> float:
    """|phi_CORDIC - atan2| <= residual rotation + table rounding + shift truncation (radius r_q in fixed-point units)."""
    n = fe.cordic_iterations
    return math.degrees(math.atan(2.0 ** -(n - 1))) + n * 2.0 ** -fe.phi_frac_bits \
        + math.degrees(2.0 * n * 2.0 ** -fe.cordic_guard_bits / max(r_q, 1.0))


def rint_even(x: float) -> int:
    return round(x)     # Python: ties to even, exact


def slice_fill(x, y, z, t, fe: FrontEnd):
    """O11 + O12 for the hits of ONE fill (arrays in input order).
    Returns (u [M] fp32, v [M] fp32, src [M] int64 indices into the fill's arrays, counts [windows_per_fill])."""
    st = float(2 ** fe.time_frac_bits)
    t0q, sq, wq = D._llround(fe.t0 * st), D._llround(fe.step * st), D._llround(fe.width * st)
    assert sq >= 1 and wq >= 1
    sx = float(2 ** fe.xy_frac_bits)
    per_window: List[List[Tuple[np.float32, np.float32, int]]] = [[] for _ in range(fe.windows_per_fill)]
    for i in range(len(x)):
        xf, yf, zf, tf = (float(np.float32(a[i])) for a in (x, y, z, t))
        if not all(math.isfinite(a) for a in (xf, yf, zf, tf)):
            continue
        if abs(xf) > fe.xy_max or abs(yf) > fe.xy_max or abs(tf * st) >= 2.0 ** 31:
            continue
        xq, yq = rint_even(xf * sx), rint_even(yf * sx)
        if xq == 0 and yq == 0:
            continue
        d = rint_even(tf * st) - t0q
        w_hi = d // sq                          # floor
        w_lo = (d - wq) // sq + 1
        phi = np.float32(cordic_phi_q(xq, yq, fe) * 2.0 ** -fe.phi_frac_bits)      # exact: |phi_q| < 2^24
        for w in range(max(w_lo, 0), min(w_hi, fe.windows_per_fill - 1) + 1):
            per_window[w].append((phi, np.float32(zf), i))
    u = np.array([h[0] for w in per_window for h in w], np.float32)
    v = np.array([h[1] for w in per_window for h in w], np.float32)
    src = np.array([h[2] for w in per_window for h in w], np.int64)
    return u, v, src, np.array([len(w) for w in per_window], np.int64)


def slice_batch(x, y, z, t, fill_offsets, fe: FrontEnd):
    """O11 over a batch of fills: (u, v, src [global input index], offsets [n_fills * windows_per_fill + 1])."""
    us, vs, ss, counts = [], [], [], []
    for f in range(len(fill_offsets) - 1):
        a, b = int(fill_offsets[f]), int(fill_offsets[f + 1])
        u, v, s, c = slice_fill(x[a:b], y[a:b], z[a:b], t[a:b], fe)
        us.append(u); vs.append(v); ss.append(s + a); counts.append(c)
    cat = lambda xs, dt: np.concatenate(xs).astype(dt) if xs else np.zeros(0, dt)
    offsets = np.concatenate([[0], np.cumsum(cat(counts, np.int64))]).astype(np.int64)
    return cat(us, np.float32), cat(vs, np.float32), cat(ss, np.int64), offsets


# ----------------------------------------------------------------------------- O13 peel-off
def peel_event(u: Sequence, v: Sequence, p: D.Params) -> Tuple[List[Tuple[int, int, int]], np.ndarray]:
    """B7: iterative global-maximum track finding.  Returns ([(theta_bin, rho_bin, votes)] in order found, labels [N])."""
    k = D.constants(p)
    n = len(u)
    labels = -np.ones(n, np.int32)
    hits = [D.quantise_hit(u[i], v[i], p, k) for i in range(n)]
    alive = [h[0] for h in hits]
    half = 2 ** (k.F - 1) if k.F >= 1 else 0
    tracks = []
    while len(tracks) < p.max_candidates:
        acc = np.zeros((p.n_theta, p.n_rho), np.int64)
        for i in range(n):
            if not alive[i]:
                continue
            for tt in range(p.n_theta):
                r = D.fixed_point_rho(hits[i][1], hits[i][2], tt, k) // 2 ** k.F
                if 0 <= r < p.n_rho:
                    acc[tt, r] += 1
        L = int(np.argmax(acc))                    # first occurrence of the maximum = lowest linear index
        tb, rb = divmod(L, p.n_rho)
        if acc[tb, rb] < p.vote_threshold:
            break
        slot = len(tracks)
        removed = 0
        for i in range(n):
            if alive[i]:
                e = D.fixed_point_rho(hits[i][1], hits[i][2], tb, k) - (rb * 2 ** k.F + half)
                if abs(e) <= k.Wq:
                    labels[i] = slot
                    alive[i] = False
                    removed += 1
        if removed == 0:                           # a window narrower than half a bin can miss every voter: no progress, stop
            break
        tracks.append((tb, rb, int(acc[tb, rb])))
    return tracks, labels


# ----------------------------------------------------------------------------- O14 two-stage (coarse -> fine) Hough
def two_stage_event(u: Sequence, v: Sequence, p: D.Params, c_theta: int, c_rho: int) -> Tuple[List[Tuple[int, int, int]], int]:
    """B8.  Returns ([(theta_bin, rho_bin, votes)] ranked by (votes desc, linear index asc), n_found)."""
    k = D.constants(p)
    two_f = 2 ** k.F
    nT, nR = -(-p.n_theta // c_theta), -(-p.n_rho // c_rho)
    hits = [h for h in (D.quantise_hit(u[i], v[i], p, k) for i in range(len(u))) if h[0]]
    coarse = np.zeros((nT, nR), np.int64)
    for _, uq, vq in hits:
        for T in range(nT):
            t = min(T * c_theta + c_theta // 2, p.n_theta - 1)
            r = D.fixed_point_rho(uq, vq, t, k) // two_f
            if 0 <= r < p.n_rho:
                coarse[T, r // c_rho] += 1
    pc = D.Params(nT, nR, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window, p.max_candidates, p.hit_frac_bits, k.F)
    cpk = D.peaks(coarse, pc)
    cpk.sort(key=lambda b: (-int(coarse[b]), b[0] * nR + b[1]))
    found = {}
    for (T, R) in cpk[: p.max_candidates]:
        t0, t1 = max(0, (T - 1) * c_theta), min(p.n_theta, (T + 2) * c_theta)
        r0, r1 = max(0, (R - 1) * c_rho), min(p.n_rho, (R + 2) * c_rho)
        patch = np.zeros((t1 - t0, r1 - r0), np.int64)
        for _, uq, vq in hits:
            for t in range(t0, t1):
                r = D.fixed_point_rho(uq, vq, t, k) // two_f
                if r0 <= r < r1:
                    patch[t - t0, r - r0] += 1
        best = None
        for t in range(t0, t1):
            for r in range(r0, r1):
                key = (int(patch[t - t0, r - r0]), -(t * p.n_rho + r))
                if best is None or key > best:
                    best = key
        if best is not None and best[0] >= p.vote_threshold:
            L = -best[1]
            found[L] = best[0]
    ranked = sorted(found.items(), key=lambda kv: (-kv[1], kv[0]))
    return [(L // p.n_rho, L % p.n_rho, c) for L, c in ranked], len(ranked)
