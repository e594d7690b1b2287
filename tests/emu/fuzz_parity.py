"""Random plans and random events through the kernels in the host model against the oracle -- a long-running companion of
tests/test_emulated_kernels.py (TEST INFRASTRUCTURE; not part of the pytest suite).

    python tests/emu/fuzz_parity.py --cases 200 --seed 1

Per case: a random grid (any n_theta, n_rho; power-of-two or not), rho range, coordinate limit, H, threshold, K, window, counter
type, a few events mixing collinear groups, uniform noise, duplicates, out-of-range and non-finite hits; fast / small-lists /
general-only plan; a random thread schedule.  Compares accumulators, digests, n_found, records and labels bit for bit.
"""
import argparse
import math
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, os.path.join(ROOT, "tests"), HERE):
    if p not in sys.path:
        sys.path.insert(0, p)

import hough_emu as E  # noqa: E402
from oracle import hough_c as C  # noqa: E402
from oracle import hough_def as D  # noqa: E402


def random_case(rng):
    n_theta = int(rng.choice([rng.integers(1, 40), rng.integers(40, 300), rng.choice([64, 128, 180, 256, 512])]))
    n_rho = int(rng.choice([rng.integers(1, 40), rng.integers(40, 700), rng.choice([64, 128, 256, 512, 1000, 1024])]))
    if n_theta * n_rho > 300000:
        n_theta = max(1, 300000 // n_rho)
    coord = float(rng.choice([1.0, 50.0, 256.0, 400.0, 1000.0]))
    H = int(rng.choice([0, 3, 6, 6, 6, 8]))
    if coord * 2 ** H > 70000:
        H = 6 if coord <= 1000 else 3
    half = coord * float(rng.choice([0.4, 1.0, 1.45, 3.0]))
    shift = float(rng.choice([0.0, 0.0, 0.3 * half, -0.2 * half]))
    rho_min, rho_max = -half + shift, half + shift
    T = int(rng.choice([1, 2, 3, 5, 8, 20]))
    K = int(rng.choice([1, 3, 8, 16, 128, 128, 1000, 2000]))
    d_rho = (rho_max - rho_min) / n_rho
    w = d_rho * float(rng.choice([0.0, 0.3, 1.0, 1.0, 2.5, 40.0]))
    lo, hi = 0.0, math.pi
    if rng.random() < 0.2:
        lo = float(rng.uniform(0, 2)); hi = lo + float(rng.uniform(0.2, 3.0))
    # theta wrap (reading B9) wherever the seam closes: default window, symmetric rho range, three or more rows
    wrap = bool(lo == 0.0 and hi == math.pi and shift == 0.0 and n_theta >= 3 and rng.random() < 0.5)
    p = D.Params(n_theta, n_rho, rho_min, rho_max, coord, T, w, K, H, -1, lo, hi, wrap)
    try:
        D.constants(p)
        if D.default_frac_bits(p) < 1:
            return None
    except AssertionError:
        return None
    n_events = int(rng.integers(1, 6))
    us, vs, offs = [], [], [0]
    for e in range(n_events):
        kind = rng.random()
        parts_u, parts_v = [], []
        if kind < 0.1:
            pass                                                      # empty event
        else:
            for _ in range(int(rng.integers(0, 5))):                  # collinear groups
                n = int(rng.integers(2, 60))
                uu = rng.uniform(-coord, coord, n) * 0.9
                m, c = rng.uniform(-2, 2), rng.uniform(-coord, coord) * 0.5
                if wrap and rng.random() < 0.5:                       # a near-vertical group: its ridge crosses the theta seam
                    vv = rng.uniform(-coord, coord, n) * 0.9
                    parts_v.append(vv); parts_u.append(np.clip(c + rng.uniform(-0.05, 0.05) * vv, -coord, coord))
                    continue
                parts_u.append(uu); parts_v.append(np.clip(m * uu + c, -coord, coord))
            n_noise = int(rng.choice([0, 5, 40, 300, 1500]))
            parts_u.append(rng.uniform(-coord, coord, n_noise)); parts_v.append(rng.uniform(-coord, coord, n_noise))
            if rng.random() < 0.3:
                n = int(rng.integers(2, 200))
                parts_u.append(np.full(n, rng.uniform(-coord, coord) * 0.5)); parts_v.append(np.full(n, rng.uniform(-coord, coord) * 0.5))
            if rng.random() < 0.3:
                parts_u.append(np.array([np.nan, np.inf, coord, -coord, coord * 1.0001])); parts_v.append(np.array([0.0, 1.0, coord, -coord, 0.0]))
        u = np.concatenate(parts_u).astype(np.float32) if parts_u else np.zeros(0, np.float32)
        v = np.concatenate(parts_v).astype(np.float32) if parts_v else np.zeros(0, np.float32)
        if rng.random() < 0.5 and len(u):
            u = np.round(u * 4) / 4                                    # coordinates on fixed-point ties and bin edges
        pm = rng.permutation(len(u))
        us.append(u[pm].astype(np.float32)); vs.append(v[pm].astype(np.float32)); offs.append(offs[-1] + len(u))
    return p, np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cases", type=int, default=100)
    ap.add_argument("--seed", type=int, default=1)
    a = ap.parse_args()
    rng = np.random.default_rng(a.seed)
    done = bad = 0
    paths = {"fast": 0, "general": 0, "deferred": 0, "wrap": 0}
    while done < a.cases:
        case = random_case(rng)
        if case is None:
            continue
        p, u, v, offsets = case
        flags = int(rng.choice([0, 0, E.FLAG_SMALL_LISTS, E.FLAG_GENERAL_ONLY]))
        dt = E.HOUGH_U16 if (rng.random() < 0.5 and (len(u) == 0 or np.diff(offsets).max() <= 65535)) else E.HOUGH_I32
        E.configure(seed=int(rng.integers(1, 1 << 30)), preempt_per_1024=int(rng.choice([0, 0, 16, 200])), workers=int(rng.choice([1, 1, 3])))
        try:
            o = C.run_batch(u, v, offsets, p, want_digest=True, want_acc=True)
        except RuntimeError:
            continue                                                   # the oracle rejects the plan (int32 bound)
        L = E.lib()
        g = E.run(p, u, v, offsets, dt, flags=flags)
        ok = (g["emu_violations"] == 0 and g["bounds_violations"] == 0 and g["status"] == 0 and (g["acc"] == o["acc"]).all()
              and (g["digest"] == o["digest"]).all() and (g["n_found"] == o["n_found"]).all() and (g["labels"] == o["labels"]).all())
        for e in range(len(offsets) - 1):
            k = min(int(o["n_found"][e]), p.max_candidates)
            ok = ok and g["cands"][e, :k].tobytes() == o["cands"][e, :k].tobytes()
        done += 1
        paths["fast" if g["info"]["fast_groups"] else "general"] += 1
        paths["deferred"] += g["deferred"]
        paths["wrap"] += int(p.theta_wrap)
        if not ok:
            bad += 1
            print("MISMATCH", p, "flags", flags, "dtype", dt, "hits", len(u), "offsets", offsets.tolist(),
                  "viol", g["emu_violations"], g["bounds_violations"], g["bounds_site"], g["status"], flush=True)
    print(f"fuzz seed {a.seed}: {done} cases, {bad} mismatches; plans with a fast kernel {paths['fast']}, without {paths['general']}, "
          f"events handed over {paths['deferred']}, theta-wrap plans {paths['wrap']}")
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
