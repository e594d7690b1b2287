"""Seeded synthetic pile-up events (inputs only -- none of the method's arithmetic lives here).

Stand-in for the paper's g2esoft/Geant4 pile-up samples (10 ns windows at
0.06 / 0.6 / 6 tracks/ns), which are not available.  The structure follows the paper: straight
lines in the 2-D projection plane (Sec. 4), hits on discrete detector planes (L72),
several tracks piled up per window (L72, L100), ghost/noise hits (L150).  The recipe is the one of
SURVEY.md Sec. 8(d) and DESIGN.md "Input recipe"; the five workloads mirror BASELINE.json `configs`.

This module is the only code shared by the CPU oracle's tests and the CUDA path's tests/bench: it
produces fp32 hit arrays and int64 event offsets and knows nothing about Hough space.

Draw order per chunk of CHUNK_EVENTS events (numpy Generator(PCG64(SeedSequence([SEED, cfg, cell, chunk])))):
  1. n_tracks[e]          integers in [lo, hi]            (only drawn when lo < hi)
  2. m[track]             uniform(-1, 1)
  3. c[track]             uniform(-100, 100)   [mm]
  4. smear[track, plane]  normal(0, sigma)     [mm]
  5. keep[track, plane]   random() >= inefficiency        (always drawn)
  6. noise u              uniform(-94, 94), then noise v  uniform(-194, 194)
  7. shuffle key per hit  random(); hits are ordered by (event, key)
All arithmetic in fp64, cast to fp32 at the end.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

import numpy as np

SEED = 251102742
CHUNK_EVENTS = 1000
N_PLANES = 48
PLANE_U0 = -94.0
PLANE_PITCH = 4.0
NOISE_U = 94.0
NOISE_V = 194.0

# grid / plan constants shared by all BASELINE configs
RHO_MIN = -256.0
RHO_MAX = 256.0
COORD_MAX = 256.0
HIT_FRAC_BITS = 6
MAX_CANDIDATES = 128


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config (or one cell of config 4)."""
    name: str
    cfg: int
    cell: int                      # RNG stream selector (config 4: index of the hits/event value)
    n_events: int
    tracks: Tuple[int, int]        # inclusive range of tracks per event
    sigma: float                   # Gaussian smearing of v [mm]
    noise_frac: float              # noise hits = floor(noise_frac * 48 * n_tracks + 0.5)
    inefficiency: float            # per-plane probability that a track hit is dropped
    hits_total: Optional[int]      # config 4: noise fills the event to exactly this many hits
    n_theta: int
    n_rho: int
    vote_threshold: int
    count_dtype: str               # "i32" | "u16": logical dtype of dumped accumulators
    rho_min: float = RHO_MIN
    rho_max: float = RHO_MAX
    coord_max: float = COORD_MAX
    hit_frac_bits: int = HIT_FRAC_BITS
    max_candidates: int = MAX_CANDIDATES
    assign_window_bins: float = 1.0   # w = assign_window_bins * d_rho
    # detector geometry of the generator (defaults: the 48 planes of SURVEY.md Sec. 8(d))
    n_planes: int = N_PLANES
    plane_u0: float = PLANE_U0
    plane_pitch: float = PLANE_PITCH
    noise_u: float = NOISE_U
    noise_v: float = NOISE_V

    @property
    def hits_per_event_nominal(self) -> float:
        if self.hits_total is not None:
            return float(self.hits_total)
        n_tr = 0.5 * (self.tracks[0] + self.tracks[1])
        return n_tr * self.n_planes * (1.0 - self.inefficiency) + np.floor(self.noise_frac * self.n_planes * n_tr + 0.5)

    @property
    def d_rho(self) -> float:
        return (self.rho_max - self.rho_min) / self.n_rho

    @property
    def assign_window(self) -> float:
        return self.assign_window_bins * self.d_rho

    @property
    def n_chunks(self) -> int:
        return (self.n_events + CHUNK_EVENTS - 1) // CHUNK_EVENTS

    def with_events(self, n_events: int) -> "Workload":
        return replace(self, n_events=n_events)


CFG4_HITS = (100, 500, 2000, 8000)
CFG4_GRIDS = (128, 256, 512, 1024)


def workload(cfg: int, hits_idx: int = 0, grid_idx: int = 0) -> Workload:
    """BASELINE.json configs[cfg]; for cfg 4, the cell (hits/event index, grid index)."""
    if cfg == 0:
        return Workload("cfg0_single_event_3tracks", 0, 0, 1, (3, 3), 0.1, 0.10, 0.0, None, 180, 256, 24, "i32")
    if cfg == 1:
        return Workload("cfg1_1k_events_pileup5", 1, 0, 1000, (5, 5), 0.1, 0.20, 0.0, None, 256, 256, 24, "i32")
    if cfg == 2:
        return Workload("cfg2_10k_events_pileup10to20", 2, 0, 10000, (10, 20), 0.1, 0.30, 0.05, None, 256, 512, 20, "i32")
    if cfg == 3:
        return Workload("cfg3_100k_events_pileup40", 3, 0, 100000, (40, 40), 0.15, 0.50, 0.05, None, 512, 512, 20, "u16")
    if cfg == 4:
        h = CFG4_HITS[hits_idx]
        g = CFG4_GRIDS[grid_idx]
        n_tr = max(1, int(np.floor(h / 96.0 + 0.5)))
        # threshold "0.4 x planes" = round(19.2) = 19 (reading A17)
        return Workload(f"cfg4_sweep_h{h}_g{g}", 4, hits_idx, 50000, (n_tr, n_tr), 0.1, 0.0, 0.0, h, g, g, 19, "i32")
    if cfg == 5:
        # The paper's own CPU grid (180 theta bins over 0-180 deg, 1000 rho bins over -500...500) with the
        # detector's 40 vanes as planes in phi (L72; 9 degrees apart), z within +-200 mm, 10-30 tracks per 10 ns window
        # (L156: up to 6 tracks / ns).  Not a BASELINE config: SURVEY.md 8(f) NEXT-4 "the paper's own 180 x 1000 workload".
        return Workload("paper_grid_180x1000_40vanes", 5, 0, 20000, (10, 30), 0.1, 0.30, 0.05, None, 180, 1000, 16, "u16",
                        rho_min=-500.0, rho_max=500.0, coord_max=360.0, n_planes=40, plane_u0=-175.5, plane_pitch=9.0,
                        noise_u=180.0, noise_v=200.0)
    raise ValueError(f"unknown config {cfg}")


@dataclass
class EventBatch:
    """SoA hits of a contiguous range of events."""
    u: np.ndarray            # float32 [N]
    v: np.ndarray            # float32 [N]
    offsets: np.ndarray      # int64 [n_events + 1], offsets[0] == 0
    first_event: int = 0
    truth_track: Optional[np.ndarray] = None     # int32 [N]: track index within the event, -1 = noise
    track_m: Optional[np.ndarray] = None         # float64 [n_tracks_total]
    track_c: Optional[np.ndarray] = None         # float64 [n_tracks_total]
    track_offsets: Optional[np.ndarray] = None   # int64 [n_events + 1]

    @property
    def n_events(self) -> int:
        return len(self.offsets) - 1

    @property
    def n_hits(self) -> int:
        return int(self.offsets[-1])

    def event(self, e: int):
        a, b = int(self.offsets[e]), int(self.offsets[e + 1])
        return self.u[a:b], self.v[a:b]

    def slice(self, e0: int, e1: int) -> "EventBatch":
        a, b = int(self.offsets[e0]), int(self.offsets[e1])
        tb = None
        if self.track_offsets is not None:
            ta, tbb = int(self.track_offsets[e0]), int(self.track_offsets[e1])
            tb = (self.track_m[ta:tbb], self.track_c[ta:tbb], self.track_offsets[e0:e1 + 1] - ta)
        return EventBatch(self.u[a:b], self.v[a:b], self.offsets[e0:e1 + 1] - a, self.first_event + e0,
                          None if self.truth_track is None else self.truth_track[a:b],
                          None if tb is None else tb[0], None if tb is None else tb[1],
                          None if tb is None else tb[2])

    def sha256(self) -> str:
        h = hashlib.sha256()
        h.update(np.ascontiguousarray(self.u).tobytes())
        h.update(np.ascontiguousarray(self.v).tobytes())
        h.update(np.ascontiguousarray(self.offsets).tobytes())
        return h.hexdigest()


def _rng(wl: Workload, chunk: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([SEED, wl.cfg, wl.cell, chunk])))


def generate_chunk(wl: Workload, chunk: int) -> EventBatch:
    """Events [chunk*CHUNK_EVENTS, min((chunk+1)*CHUNK_EVENTS, n_events)) of a workload."""
    e0 = chunk * CHUNK_EVENTS
    n_ev = min(CHUNK_EVENTS, wl.n_events - e0)
    if n_ev <= 0:
        raise ValueError("chunk beyond the workload")
    rng = _rng(wl, chunk)
    lo, hi = wl.tracks
    if hi > lo:
        n_tr = rng.integers(lo, hi + 1, size=n_ev).astype(np.int64)
    else:
        n_tr = np.full(n_ev, lo, dtype=np.int64)
    n_tracks = int(n_tr.sum())
    m = rng.uniform(-1.0, 1.0, size=n_tracks)
    c = rng.uniform(-100.0, 100.0, size=n_tracks)
    smear = rng.normal(0.0, wl.sigma, size=(n_tracks, wl.n_planes))
    keep = rng.random(size=(n_tracks, wl.n_planes)) >= wl.inefficiency
    planes = wl.plane_u0 + wl.plane_pitch * np.arange(wl.n_planes, dtype=np.float64)
    v_tr = m[:, None] * planes[None, :] + c[:, None] + smear
    u_tr = np.broadcast_to(planes[None, :], v_tr.shape)
    if wl.hits_total is not None:
        n_noise = wl.hits_total - wl.n_planes * n_tr
        if (n_noise < 0).any():
            raise ValueError("hits_total smaller than the track hits")
    else:
        n_noise = np.floor(wl.noise_frac * wl.n_planes * n_tr + 0.5).astype(np.int64)
    nn = int(n_noise.sum())
    nu = rng.uniform(-wl.noise_u, wl.noise_u, size=nn)
    nv = rng.uniform(-wl.noise_v, wl.noise_v, size=nn)

    ev_of_track = np.repeat(np.arange(n_ev, dtype=np.int64), n_tr)
    track_in_event = np.arange(n_tracks, dtype=np.int64) - np.repeat(np.cumsum(n_tr) - n_tr, n_tr)
    kf = keep.ravel()
    ev_th = np.repeat(ev_of_track, wl.n_planes)[kf]
    tid_th = np.repeat(track_in_event, wl.n_planes)[kf]
    ev_all = np.concatenate([ev_th, np.repeat(np.arange(n_ev, dtype=np.int64), n_noise)])
    u_all = np.concatenate([u_tr.ravel()[kf], nu])
    v_all = np.concatenate([v_tr.ravel()[kf], nv])
    t_all = np.concatenate([tid_th, np.full(nn, -1, dtype=np.int64)])
    key = rng.random(size=len(ev_all))
    order = np.lexsort((key, ev_all))
    counts = np.bincount(ev_all, minlength=n_ev).astype(np.int64)
    offsets = np.zeros(n_ev + 1, dtype=np.int64)
    np.cumsum(counts, out=offsets[1:])
    tr_off = np.zeros(n_ev + 1, dtype=np.int64)
    np.cumsum(n_tr, out=tr_off[1:])
    return EventBatch(u_all[order].astype(np.float32), v_all[order].astype(np.float32), offsets, e0,
                      t_all[order].astype(np.int32), m, c, tr_off)


def concat(batches) -> EventBatch:
    batches = list(batches)
    if len(batches) == 1:
        return batches[0]
    offs = [np.zeros(1, dtype=np.int64)]
    toffs = [np.zeros(1, dtype=np.int64)]
    base = 0
    tbase = 0
    for b in batches:
        offs.append(b.offsets[1:] + base)
        base += b.n_hits
        toffs.append(b.track_offsets[1:] + tbase)
        tbase += int(b.track_offsets[-1])
    return EventBatch(np.concatenate([b.u for b in batches]), np.concatenate([b.v for b in batches]),
                      np.concatenate(offs), batches[0].first_event,
                      np.concatenate([b.truth_track for b in batches]),
                      np.concatenate([b.track_m for b in batches]), np.concatenate([b.track_c for b in batches]),
                      np.concatenate(toffs))


def generate(wl: Workload, first_event: int = 0, n_events: Optional[int] = None) -> EventBatch:
    """Events [first_event, first_event + n_events) of a workload (any range; whole chunks are generated and sliced)."""
    if n_events is None:
        n_events = wl.n_events - first_event
    last = first_event + n_events
    if first_event < 0 or last > wl.n_events or n_events < 0:
        raise ValueError("event range outside the workload")
    if n_events == 0:
        return EventBatch(np.zeros(0, np.float32), np.zeros(0, np.float32), np.zeros(1, np.int64), first_event,
                          np.zeros(0, np.int32), np.zeros(0), np.zeros(0), np.zeros(1, np.int64))
    c0, c1 = first_event // CHUNK_EVENTS, (last - 1) // CHUNK_EVENTS
    full = concat(generate_chunk(wl, c) for c in range(c0, c1 + 1))
    return full.slice(first_event - c0 * CHUNK_EVENTS, last - c0 * CHUNK_EVENTS)


def ideal_track(m: float, c: float) -> Tuple[np.ndarray, np.ndarray]:
    """The 48 unsmeared plane hits of the line v = m*u + c (fp32), for closed-form pins."""
    planes = PLANE_U0 + PLANE_PITCH * np.arange(N_PLANES, dtype=np.float64)
    return planes.astype(np.float32), (m * planes + c).astype(np.float32)
