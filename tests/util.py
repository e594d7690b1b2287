"""Helpers shared by the tests (no method arithmetic)."""
import os

import numpy as np

from oracle import hough_def as D
from paper_2511_02742_b200 import synth

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def params_of(wl, **over) -> D.Params:
    """Oracle parameters of a synth.Workload."""
    kw = dict(n_theta=wl.n_theta, n_rho=wl.n_rho, rho_min=wl.rho_min, rho_max=wl.rho_max, coord_max=wl.coord_max,
              vote_threshold=wl.vote_threshold, assign_window=wl.assign_window, max_candidates=wl.max_candidates,
              hit_frac_bits=wl.hit_frac_bits, acc_frac_bits=-1)
    kw.update(over)
    return D.Params(**kw)


def std_params(n_theta=256, n_rho=256, T=24, K=128, w_bins=1.0, **over) -> D.Params:
    """The grid of SURVEY.md Sec. 8(d): rho in [-256, 256) mm, coord_max 256, H = 6."""
    d_rho = 512.0 / n_rho
    kw = dict(n_theta=n_theta, n_rho=n_rho, rho_min=-256.0, rho_max=256.0, coord_max=256.0, vote_threshold=T,
              assign_window=w_bins * d_rho, max_candidates=K, hit_frac_bits=6, acc_frac_bits=-1)
    kw.update(over)
    return D.Params(**kw)


def read_golden_table(name):
    """Whitespace-separated rows of a golden text fixture; '#' starts a comment."""
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows


def cands_as_tuples(cands):
    """(theta_bin, rho_bin, votes, cluster_root, cluster_nbins) per record, for numpy records or def-oracle Candidates."""
    out = []
    for c in cands:
        if hasattr(c, "theta_bin"):
            out.append((int(c.theta_bin), int(c.rho_bin), int(c.votes), int(c.cluster_root), int(c.cluster_nbins)))
        else:
            out.append((int(c["theta_bin"]), int(c["rho_bin"]), int(c["votes"]), int(c["cluster_root"]), int(c["cluster_nbins"])))
    return out


def mixed_batch(cfg, n_events, seed, long_hits=0):
    """Generator events with special ones interleaved: empty events, an event whose hits all coincide 1100 times (a bin count
    above 1023: the fast kernel must hand it over), all-invalid events, and optionally one event of `long_hits` hits."""
    wl = synth.workload(cfg)
    wl = wl.with_events(max(wl.n_events, n_events))      # more events than the config lists: further chunks of the same stream
    b = synth.generate(wl, 0, n_events)
    rng = np.random.default_rng(seed)
    us, vs, offs, kinds = [], [], [0], []
    for e in range(n_events):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        roll = rng.random()
        if roll < 0.05:
            uu, vv, kind = np.zeros(0, np.float32), np.zeros(0, np.float32), "empty"
        elif roll < 0.08:
            uu, vv, kind = np.full(1100, 7.25, np.float32), np.full(1100, -3.5, np.float32), "count>1023"
        elif roll < 0.10:
            uu, vv, kind = np.full(17, np.nan, np.float32), np.full(17, 1.0, np.float32), "invalid"
        elif long_hits and roll < 0.12:
            uu = rng.uniform(-94, 94, long_hits).astype(np.float32)
            vv = rng.uniform(-194, 194, long_hits).astype(np.float32)
            kind = "long"
        else:
            uu, vv, kind = b.u[a:z], b.v[a:z], "plain"
        us.append(uu); vs.append(vv); offs.append(offs[-1] + len(uu)); kinds.append(kind)
    return wl, np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64), kinds


def paper_grid_batch(n_events, seed=31):
    """Events on the paper's own CPU grid (180 theta bins over 0-180 deg, 1000 rho bins over -500...500) with
    40 detector planes (L72: 40 vanes): 1-8 straight tracks plus up to 200 noise hits per event.  -> (params, u, v, offsets)"""
    rng = np.random.default_rng(seed)
    p = D.Params(180, 1000, -500.0, 500.0, 360.0, 20, 1.0, 64)
    us, vs, offs = [], [], [0]
    planes = np.linspace(-195.0, 195.0, 40)
    for e in range(n_events):
        nt = int(rng.integers(1, 9))
        uu = [np.tile(planes, nt)]
        m, c = rng.uniform(-1, 1, nt), rng.uniform(-100, 100, nt)
        vv = [(m[:, None] * planes[None, :] + c[:, None] + rng.normal(0, 0.1, (nt, 40))).ravel()]
        nn = int(rng.integers(0, 200))
        uu.append(rng.uniform(-195, 195, nn)); vv.append(rng.uniform(-300, 300, nn))
        uu, vv = np.concatenate(uu).astype(np.float32), np.concatenate(vv).astype(np.float32)
        pm = rng.permutation(len(uu))
        us.append(uu[pm]); vs.append(vv[pm]); offs.append(offs[-1] + len(uu))
    return p, np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)


def synthetic_fills(n_fills, seed, hits_per_fill=600, t_span=80.0):
    """RecoHits of a few fills: points on the 40 radial vanes (r from 70 to 290 mm, z within +-200 mm), times
    uniform over the fill, some invalid ones; in no particular order."""
    rng = np.random.default_rng(seed)
    xs, ys, zs, ts, fo = [], [], [], [], [0]
    for f in range(n_fills):
        n = int(rng.integers(hits_per_fill // 2, hits_per_fill + 1)) if f != 1 else 0
        vane = rng.integers(0, 40, n)
        r = rng.uniform(70.0, 290.0, n)
        ang = np.radians(vane * 9.0 + 4.5)
        x, y = r * np.cos(ang), r * np.sin(ang)
        z, t = rng.uniform(-200, 200, n), rng.uniform(-15.0, t_span, n)
        if n > 8:
            x[3], t[5], z[6] = np.nan, np.inf, -np.inf
            x[7] = y[7] = 0.0
            x[8] = 600.0
            t[9] = 5.0                                                      # exactly on a window edge
        xs.append(x); ys.append(y); zs.append(z); ts.append(t); fo.append(fo[-1] + n)
    cat = lambda a: np.concatenate(a).astype(np.float32)
    return cat(xs), cat(ys), cat(zs), cat(ts), np.array(fo, np.int64)


def fills_with_tracks(n_fills, seed, tracks_per_fill=2):
    """RecoHits of fills that hold helix-like tracks: phi (degrees) linear in z, one hit per crossed vane, all hits of a track
    within one ns of each other (a helix projected onto the phi-z plane is a straight line)."""
    rng = np.random.default_rng(seed)
    xs, ys, zs, ts, fo = [], [], [], [], [0]
    for f in range(n_fills):
        n_f = 0
        for trk in range(tracks_per_fill):
            z0, slope, t_trk = rng.uniform(-100, 100), rng.uniform(-0.8, 0.8), rng.uniform(8, 22)
            vanes = np.arange(int(rng.integers(0, 10)), int(rng.integers(20, 40)))
            phi = np.radians(vanes * 9.0 + 4.5 - 180.0)
            r = rng.uniform(100, 280, len(vanes))
            xs.append(r * np.cos(phi)); ys.append(r * np.sin(phi)); zs.append(z0 + slope * (vanes * 9.0 - 180.0))
            ts.append(np.full(len(vanes), t_trk) + rng.uniform(-0.5, 0.5, len(vanes)))
            n_f += len(vanes)
        fo.append(fo[-1] + n_f)
    x, y, z, t = (np.concatenate(a).astype(np.float32) for a in (xs, ys, zs, ts))
    return x, y, z, t, np.array(fo, np.int64)
