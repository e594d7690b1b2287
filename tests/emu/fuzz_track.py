"""Random front-end grids / fills and random refit geometries through the kernels in the host model against oracle/track_def.py
(TEST INFRASTRUCTURE; not part of the pytest suite).

    python tests/emu/fuzz_track.py --cases 100 --seed 1
"""
import argparse
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
from oracle import track_def as T  # noqa: E402


def front_case(rng):
    step = float(rng.choice([5.0, 2.5, 1.0, 7.25, 0.5]))
    width = float(rng.choice([10.0, step, 2 * step, 3.5 * step, 0.4 * step]))
    fe = T.FrontEnd(t0=float(rng.choice([0.0, -12.5, 100.0, 3.00390625])), width=width, step=step,
                    windows_per_fill=int(rng.integers(1, 40)), xy_max=float(rng.choice([512.0, 300.0, 64.0])))
    n_fills = int(rng.integers(1, 7))
    xs, ys, zs, ts, fo = [], [], [], [], [0]
    span = fe.t0 + fe.step * fe.windows_per_fill + fe.width
    for f in range(n_fills):
        n = int(rng.choice([0, 1, 31, 32, 33, 200, 1500]))
        x = rng.uniform(-1.1, 1.1, n) * fe.xy_max
        y = rng.uniform(-1.1, 1.1, n) * fe.xy_max
        z = rng.uniform(-200, 200, n)
        t = rng.uniform(fe.t0 - 2 * fe.width, span + fe.width, n)
        if rng.random() < 0.5:
            t = np.round(t / fe.step * 2) * fe.step / 2                # times on window edges
        if rng.random() < 0.5:
            t = np.sort(t)                                              # time-ordered input, as a DAQ would deliver it
        for a in (x, y, z, t):
            if n > 4 and rng.random() < 0.3:
                a[rng.integers(0, n)] = rng.choice([np.nan, np.inf, -np.inf])
        if n > 2:
            x[0] = y[0] = 0.0
        xs.append(x); ys.append(y); zs.append(z); ts.append(t); fo.append(fo[-1] + n)
    cat = lambda a: np.concatenate(a).astype(np.float32)
    return fe, cat(xs), cat(ys), cat(zs), cat(ts), np.array(fo, np.int64)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cases", type=int, default=100)
    ap.add_argument("--seed", type=int, default=1)
    a = ap.parse_args()
    rng = np.random.default_rng(a.seed)
    bad = 0
    for case in range(a.cases):
        E.configure(seed=int(rng.integers(1, 1 << 30)), preempt_per_1024=int(rng.choice([0, 50])), workers=int(rng.choice([1, 3])))
        fe, x, y, z, t, fo = front_case(rng)
        ou, ov, osrc, ooff = T.slice_batch(x, y, z, t, fo, fe)
        g = E.frontend_slice(fe, x, y, z, t, fo)
        M = int(ooff[-1])
        ok = (g["status"] == 0 and (g["offsets"] == ooff).all() and (g["src"][:M] == osrc).all()
              and g["u"][:M].tobytes() == ou.tobytes() and g["v"][:M].tobytes() == ov.tobytes())
        # refit on the sliced windows: labels from the oracle's one-pass search on a coarse grid
        if ok and M > 0:
            p = D.Params(int(rng.choice([16, 45, 64])), int(rng.choice([32, 100, 128])), -512.0, 512.0, 512.0, int(rng.choice([2, 4])),
                         float(rng.choice([8.0, 32.0])), int(rng.choice([1, 4, 16])))
            o = C.run_batch(ou, ov, ooff, p)
            geom = T.PlaneGeometry(origin=float(rng.choice([-180.0, -175.5, 0.0])), pitch=float(rng.choice([9.0, 4.0, 0.25, 33.0])),
                                   n_planes=int(rng.choice([1, 5, 40, 64])), min_run=int(rng.choice([1, 3, 5])), wrap=bool(rng.random() < 0.5))
            fits, rc = E.refit(p, ou, ov, ooff, o["n_found"], o["labels"], geom)
            ok = ok and rc == 0
            for e in range(len(ooff) - 1):
                aa, zz = int(ooff[e]), int(ooff[e + 1])
                nk = min(int(o["n_found"][e]), p.max_candidates)
                for s, f in enumerate(T.refit_event(ou[aa:zz], ov[aa:zz], o["labels"][aa:zz], nk, p, geom)):
                    r = fits[e, s]
                    ok = ok and (int(r["n_hits"]), int(r["plane_mask"]), int(r["max_run"]), int(r["flags"])) == (f.n_hits, f.plane_mask, f.max_run, f.flags) \
                        and r["slope"].tobytes() == f.slope.tobytes() and r["intercept"].tobytes() == f.intercept.tobytes()
        if not ok:
            bad += 1
            print("MISMATCH case", case, fe, "fills", fo.tolist(), flush=True)
    print(f"fuzz_track seed {a.seed}: {a.cases} cases, {bad} mismatches")
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
