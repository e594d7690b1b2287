"""Helpers shared by the tests (no method arithmetic)."""
import os

import numpy as np

from oracle import hough_def as D

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
