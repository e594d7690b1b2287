"""Definition oracle: Hough track finding written out with Python integers, one step per function.

TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It shares no code with the CUDA path
(paper_2511_02742_b200/csrc, include/hough.h) and never imports it.

What it computes (per event, independently), with the passage each step follows:

  O1 quantise   hit validity and fixed-point coordinates            DESIGN.md reading A4/A5/A14
  O2 constants  F, M, cos/sin tables by formula, offset, window     DESIGN.md reading A2/A4
  O3 vote       rho = phi cos(theta) + z sin(theta)                 PAPER.md L90-92, Eq. 4.1
                2-D histogram, theta in [0,180 deg), floor binning  PAPER.md L106 (Sec. 5)
                "each hit contributes to multiple bins"
  O4 peaks      "bin with the highest number of entries"            PAPER.md L94, L106; generalised to
                all strict local maxima >= threshold                BASELINE.json north_star, reading A7
  O5 clusters   8-connected components of the thresholded mask      PAPER.md L29 keyword "cluster finding",
                                                                    reading A7
     (option theta_wrap, reading B9: O4 and O5 on the neighbourhood that continues past the theta seam -- the line
      (theta + pi, rho) is the line (theta, -rho), Eq. 4.1; pinned by P9w, brute force on the unrolled theta axis)
  O6 rank       order by (votes desc, index asc), keep K            reading A8/A11
  O7 assign     "selecting the hits that align with the straight    PAPER.md L106, L94; reading A12/A13
                line formed by the identified (theta, rho)"
  O8 digest     order-independent 64-bit checksum of an accumulator debug aid, DESIGN.md

Everything after O1 is integer arithmetic on unbounded Python ints; the int32 no-overflow bound that the
fixed-point design promises is asserted, not assumed.  Pure Python loops: use on small inputs only
(oracle/hough_c.py is the plain C twin for the large configs; tests check the two agree).

Parity status: O1-O3, O5, O8 are pinned by closed forms / invariants / library special cases / brute force
(tests/test_oracle_pins.py).  The *choices* A2, A6-A13 (theta sampling point, >= threshold, local-maximum
definition, tie-breaks, window metric, K) are readings of a paper that is silent on them: "parity unpinned"
for those choices; this file is their normative statement.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Sequence, Tuple

import numpy as np

INT32_MAX = 2 ** 31 - 1
MASK64 = 2 ** 64 - 1


@dataclass(frozen=True)
class Params:
    n_theta: int
    n_rho: int
    rho_min: float
    rho_max: float
    coord_max: float
    vote_threshold: int
    assign_window: float          # w, in rho units
    max_candidates: int           # K
    hit_frac_bits: int = 6        # H
    acc_frac_bits: int = -1       # F; < 0 -> default formula
    theta_min: float = 0.0        # theta window [theta_min, theta_max) in radians; the paper's is [0, pi)
    theta_max: float = math.pi
    theta_wrap: bool = False      # O4 / O5 treat theta = pi as theta = 0 with rho mirrored (reading B9); default: no wrap

    def theta_of(self, t: int) -> float:
        """theta_t = theta_min + (theta_max - theta_min) t / n_theta (left bin edge); for the default window pi t / n_theta."""
        return self.theta_min + (self.theta_max - self.theta_min) * t / self.n_theta


@dataclass(frozen=True)
class Constants:
    H: int
    F: int
    d_rho: float
    M: float
    Cq: Tuple[int, ...]
    Sq: Tuple[int, ...]
    Oq: int
    Wq: int


@dataclass(frozen=True)
class Candidate:
    theta_bin: int
    rho_bin: int
    votes: int
    cluster_root: int
    cluster_nbins: int
    theta: np.float32
    rho: np.float32


def _llround(x: float) -> int:
    """C llround: nearest integer, halves away from zero."""
    ax = abs(x)
    f = math.floor(ax)
    n = int(f) + (1 if ax - f >= 0.5 else 0)      # ax - f is exact in double
    return n if x >= 0 else -n


def _tables(p: Params, F: int):
    """(M, C_q, S_q, O_q, W_q) for a given F."""
    H = p.hit_frac_bits
    d_rho = (p.rho_max - p.rho_min) / p.n_rho
    M = float(2 ** (F - H)) / d_rho if F >= H else 1.0 / (float(2 ** (H - F)) * d_rho)
    Cq = tuple(_llround(math.cos(p.theta_of(t)) * M) for t in range(p.n_theta))
    Sq = tuple(_llround(math.sin(p.theta_of(t)) * M) for t in range(p.n_theta))
    Oq = _llround(-p.rho_min * float(2 ** F) / d_rho)
    Wq = _llround(p.assign_window * float(2 ** F) / d_rho)
    return M, Cq, Sq, Oq, Wq


def int32_proof(p: Params, F: int) -> bool:
    """Every intermediate of O3 and O7 fits int32 for EVERY valid hit: q_max (max_t |C_q| + |S_q|) + |O_q| <= 2^31 - 1 with
    q_max = floor(coord_max 2^H + 1/2) >= |u_q|, |v_q| (the corner hits attain it), and (n_rho + 1) 2^F <= 2^31 - 1."""
    _, Cq, Sq, Oq, _ = _tables(p, F)
    qmax = math.floor(p.coord_max * float(2 ** p.hit_frac_bits) + 0.5)
    max_cs = max(abs(c) + abs(s) for c, s in zip(Cq, Sq))
    return qmax * max_cs + abs(Oq) <= INT32_MAX and (p.n_rho + 1) * 2 ** F <= INT32_MAX


def default_frac_bits(p: Params) -> int:
    """O2: the largest F <= 24 that keeps every intermediate inside int32.  Start from the closed form
    span * 2^F <= 2^31 - 1, span = max(sqrt(2) coord_max / d_rho + max(|rho_min|, |rho_max|) / d_rho + 2, n_rho + 1)
    (which already is the answer unless d_rho is far below the hit resolution 2^-H), then lower F until int32_proof holds."""
    d_rho = (p.rho_max - p.rho_min) / p.n_rho
    span = math.sqrt(2.0) * p.coord_max / d_rho + max(abs(p.rho_min), abs(p.rho_max)) / d_rho + 2.0
    span = max(span, float(p.n_rho + 1))
    F = 24
    while F > 0 and span * float(2 ** F) > float(INT32_MAX):
        F -= 1
    while F > 1 and not int32_proof(p, F):
        F -= 1
    return F


def constants(p: Params) -> Constants:
    """O2.  theta_t = theta_min + (theta_max - theta_min) t / n_theta (left bin edge; the paper's window [0, pi) gives
    pi t / n_theta, bit for bit);  tables by formula in double."""
    H = p.hit_frac_bits
    F = p.acc_frac_bits if p.acc_frac_bits >= 0 else default_frac_bits(p)
    d_rho = (p.rho_max - p.rho_min) / p.n_rho
    M, Cq, Sq, Oq, Wq = _tables(p, F)
    return Constants(H, F, d_rho, M, Cq, Sq, Oq, Wq)


def quantise_hit(u, v, p: Params, k: Constants) -> Tuple[bool, int, int]:
    """O1.  u, v are fp32 values.  valid <=> finite and |u|, |v| <= coord_max;
    u_q = rint(u * 2^H), ties to even (the product is exact: power-of-two scale)."""
    uf, vf = float(np.float32(u)), float(np.float32(v))
    if not (math.isfinite(uf) and math.isfinite(vf)):
        return False, 0, 0
    if abs(uf) > p.coord_max or abs(vf) > p.coord_max:
        return False, 0, 0
    s = float(2 ** k.H)
    return True, round(uf * s), round(vf * s)     # Python round(): ties to even, exact int


def fixed_point_rho(uq: int, vq: int, t: int, k: Constants) -> int:
    """O3, Eq. 4.1 in fixed point: a = (rho - rho_min) / d_rho * 2^F = u_q C_q[t] + v_q S_q[t] + O_q."""
    a = uq * k.Cq[t] + vq * k.Sq[t] + k.Oq
    assert abs(uq * k.Cq[t]) + abs(vq * k.Sq[t]) + abs(k.Oq) <= INT32_MAX, "int32 bound of the fixed-point design violated"
    return a


def vote_event(u: Sequence, v: Sequence, p: Params, k: Constants = None) -> np.ndarray:
    """O3: acc[t][r] += 1 for every valid hit and every theta bin t, r = floor(a / 2^F), dropped if outside [0, n_rho)."""
    k = k or constants(p)
    acc = np.zeros((p.n_theta, p.n_rho), dtype=np.int64)
    two_f = 2 ** k.F
    for uu, vv in zip(u, v):
        ok, uq, vq = quantise_hit(uu, vv, p, k)
        if not ok:
            continue
        for t in range(p.n_theta):
            r = fixed_point_rho(uq, vq, t, k) // two_f       # floor division (Python // floors for negatives too)
            if 0 <= r < p.n_rho:
                acc[t, r] += 1
    return acc


def _key(acc: np.ndarray, t: int, r: int, n_rho: int) -> Tuple[int, int]:
    """Strict total order on bins: (count, -linear index), linear index L = t * n_rho + r."""
    return int(acc[t, r]), -(t * n_rho + r)


_NEIGH8 = ((-1, -1), (-1, 0), (-1, 1), (0, -1), (0, 1), (1, -1), (1, 0), (1, 1))


def check_theta_wrap(p: Params) -> None:
    """Reading B9: the line (theta + pi, rho) IS the line (theta, -rho) (Eq. 4.1: cos and sin change sign together).  With the
    paper's window [0, pi) and a rho range symmetric about 0, bin (t, r) continued past the last theta row is therefore bin
    (t - n_theta, n_rho - 1 - r).  Wrap needs exactly that window and range, and n_theta >= 3 so that the row before and the
    row after a row are different rows."""
    assert p.theta_min == 0.0 and p.theta_max == math.pi and p.rho_min == -p.rho_max and p.n_theta >= 3, \
        "theta_wrap needs theta in [0, pi), rho_min = -rho_max and n_theta >= 3"


def neighbours8(t: int, r: int, p: Params) -> List[Tuple[int, int]]:
    """The in-grid 8-neighbours of bin (t, r).  Without wrap: the rectangle's.  With wrap (B9) the theta rows form a ring with
    a twist: the step from row n_theta - 1 to row 0 (and back) mirrors the rho bin, r -> n_rho - 1 - r."""
    out = []
    for dt, dr in _NEIGH8:
        tt, rr = t + dt, r + dr
        if p.theta_wrap and tt < 0:
            tt, rr = tt + p.n_theta, p.n_rho - 1 - rr
        elif p.theta_wrap and tt >= p.n_theta:
            tt, rr = tt - p.n_theta, p.n_rho - 1 - rr
        if 0 <= tt < p.n_theta and 0 <= rr < p.n_rho:
            out.append((tt, rr))
    return out


def peaks(acc: np.ndarray, p: Params) -> List[Tuple[int, int]]:
    """O4: on(b) <=> acc(b) >= T;  peak(b) <=> on(b) and key(b) > key(n) for all in-grid 8-neighbours (no wrap unless
    p.theta_wrap, reading B9: then the neighbours across the theta seam count too)."""
    if p.theta_wrap:
        check_theta_wrap(p)
    out = []
    for t in range(p.n_theta):
        for r in range(p.n_rho):
            if acc[t, r] < p.vote_threshold:
                continue
            kb = _key(acc, t, r, p.n_rho)
            if all(_key(acc, tt, rr, p.n_rho) < kb for tt, rr in neighbours8(t, r, p)):
                out.append((t, r))
    return out


def components(acc: np.ndarray, p: Params) -> Tuple[np.ndarray, List[Tuple[Tuple[int, int], int]]]:
    """O5: 8-connected components of the on-mask (no wrap unless p.theta_wrap, reading B9), by union-find.
    Returns (label array: component id per bin or -1, list per component of (root bin = max-key bin, n_bins))."""
    nt, nr = p.n_theta, p.n_rho
    if p.theta_wrap:
        check_theta_wrap(p)
    parent = {}

    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x

    on = acc >= p.vote_threshold
    for t in range(nt):
        for r in range(nr):
            if not on[t, r]:
                continue
            b = t * nr + r
            parent[b] = b
            for tt, rr in neighbours8(t, r, p):
                if tt * nr + rr < b and on[tt, rr]:                    # the neighbours already visited (smaller linear index)
                    ra, rb = find(tt * nr + rr), find(b)
                    if ra != rb:
                        parent[max(ra, rb)] = min(ra, rb)
    labels = -np.ones((nt, nr), dtype=np.int64)
    comp_of_root = {}
    comps: List[List] = []
    for b in sorted(parent):
        root = find(b)
        if root not in comp_of_root:
            comp_of_root[root] = len(comps)
            comps.append([None, 0])
        cid = comp_of_root[root]
        t, r = divmod(b, nr)
        labels[t, r] = cid
        comps[cid][1] += 1
        if comps[cid][0] is None or _key(acc, t, r, nr) > _key(acc, *comps[cid][0], nr):
            comps[cid][0] = (t, r)
    return labels, [(c[0], c[1]) for c in comps]


def find_clusters_event(acc: np.ndarray, p: Params) -> Tuple[List[Candidate], int]:
    """O4-O6: candidates in rank order (votes desc, linear index asc), truncated to K; n_found untruncated."""
    pk = peaks(acc, p)
    labels, comps = components(acc, p)
    pk.sort(key=lambda b: (-int(acc[b]), b[0] * p.n_rho + b[1]))
    n_found = len(pk)
    kept = pk[: p.max_candidates]
    slot_of = {b: s for s, b in enumerate(kept)}
    d_rho = (p.rho_max - p.rho_min) / p.n_rho
    out = []
    for (t, r) in kept:
        root_bin, n_bins = comps[labels[t, r]]
        # the root out-ranks every peak of its component, so it is kept whenever one of them is
        out.append(Candidate(t, r, int(acc[t, r]), slot_of[root_bin], n_bins,
                             np.float32(p.theta_of(t)), np.float32(p.rho_min + (r + 0.5) * d_rho)))
    return out, n_found


def assign_event(u: Sequence, v: Sequence, cands: Sequence[Candidate], p: Params, k: Constants = None) -> np.ndarray:
    """O7: label = slot of the kept candidate with minimal |e| among those with |e| <= W_q, ties -> lowest slot; else -1.
    e = a(hit, t_c) - (r_c 2^F + 2^(F-1)): signed fixed-point distance to the peak-bin-centre line, at the peak's theta."""
    k = k or constants(p)
    labels = -np.ones(len(u), dtype=np.int32)
    half = 2 ** (k.F - 1) if k.F >= 1 else 0
    for i, (uu, vv) in enumerate(zip(u, v)):
        ok, uq, vq = quantise_hit(uu, vv, p, k)
        if not ok:
            continue
        best = None
        for s, c in enumerate(cands):
            e = fixed_point_rho(uq, vq, c.theta_bin, k) - (c.rho_bin * 2 ** k.F + half)
            assert abs(e) <= INT32_MAX
            if abs(e) <= k.Wq and (best is None or abs(e) < best[0]):
                best = (abs(e), s)
        if best is not None:
            labels[i] = best[1]
    return labels


def mix64(x: int) -> int:
    """SplitMix64 finaliser of (x + golden gamma)."""
    z = (x + 0x9E3779B97F4A7C15) & MASK64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
    return z ^ (z >> 31)


def digest(acc: np.ndarray) -> int:
    """O8: D = sum_b acc(b) * mix64(L(b)) mod 2^64 (linear in acc, independent of the order of accumulation)."""
    n_rho = acc.shape[1]
    d = 0
    for t, r in zip(*np.nonzero(acc)):
        d = (d + int(acc[t, r]) * mix64(int(t) * n_rho + int(r))) & MASK64
    return d


def run_event(u, v, p: Params):
    """Whole path for one event: (acc, candidates, n_found, labels)."""
    k = constants(p)
    acc = vote_event(u, v, p, k)
    cands, n_found = find_clusters_event(acc, p)
    labels = assign_event(u, v, cands, p, k)
    return acc, cands, n_found, labels
