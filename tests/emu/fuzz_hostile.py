"""Hostile inputs through every entry point of the C ABI in the host model: what a call takes as INPUT (offsets, records, counts,
labels, fill offsets) is garbage of the right type and size.  TEST INFRASTRUCTURE; not part of the pytest suite.

    python tests/emu/fuzz_hostile.py --cases 300 --seed 1

Nothing is compared with the oracle: the only claims are the ones include/hough.h makes for caller data -- no access outside the
buffers (every "device" buffer of the model ends at an inaccessible page and the kernels' own index checks are compiled in: a
violation is counted, an overrun of a guard page kills the process, and the case number printed before each call says where),
and a return code instead of a crash.  Pointers and sizes themselves are honest: the ABI cannot check those.
"""
import argparse
import ctypes
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, os.path.join(ROOT, "tests"), HERE):
    if p not in sys.path:
        sys.path.insert(0, p)

import hough_emu as E  # noqa: E402

vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64


def garbage_offsets(rng, n_events, n_hits):
    """Starts from a valid partition and corrupts it: negative, decreasing, beyond the buffers, huge."""
    cuts = np.sort(rng.integers(0, n_hits + 1, n_events - 1)) if n_events > 1 else np.zeros(0, np.int64)
    off = np.concatenate([[0], cuts, [n_hits]]).astype(np.int64)
    for _ in range(int(rng.integers(0, 4))):
        i = int(rng.integers(0, n_events + 1))
        off[i] = int(rng.choice([-1, -2 ** 40, n_hits + 1, n_hits + 10 ** 6, 2 ** 62, 0, n_hits, int(rng.integers(0, n_hits + 1))]))
    return off


def garbage_i32(rng, n, lo, hi):
    a = rng.integers(lo, hi, n).astype(np.int32)
    for _ in range(int(rng.integers(0, 4))):
        if n:
            a[int(rng.integers(0, n))] = int(rng.choice([-1, -2 ** 31, 2 ** 31 - 1, 4096, 65535, 0]))
    return a


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cases", type=int, default=200)
    ap.add_argument("--seed", type=int, default=1)
    a = ap.parse_args()
    rng = np.random.default_rng(a.seed)
    L = E.lib()
    L.hough_refit_tracks.argtypes = [vp, vp, vp, vp, i32, vp, vp, ctypes.POINTER(E.PlaneGeometry), vp, vp]
    L.hough_find_tracks_peeloff.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp, vp]
    L.hough_find_two_stage.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, vp]
    L.hough_frontend_create.argtypes = [ctypes.POINTER(E.FrontDesc), ctypes.POINTER(vp)]
    L.hough_frontend_destroy.argtypes = [vp]
    L.hough_frontend_slice.argtypes = [vp, vp, vp, vp, vp, vp, i32, i64, vp, vp, vp, vp, i64, vp]
    bad = 0
    rcs = {}
    for case in range(a.cases):
        L.cuda_emu_reset_violations()
        E.configure(seed=int(rng.integers(1, 1 << 30)), preempt_per_1024=0, workers=int(rng.choice([1, 1, 3])))
        n_theta, n_rho = int(rng.choice([8, 45, 64, 180])), int(rng.choice([16, 64, 100, 256]))
        K, T = int(rng.choice([1, 4, 16, 128])), int(rng.choice([1, 2, 5]))
        n_events, n_hits = int(rng.integers(1, 7)), int(rng.choice([0, 1, 40, 300, 1500]))
        max_hpe = int(rng.choice([1, 50, 400, 2000]))
        dt = int(rng.choice([E.HOUGH_I32, E.HOUGH_U16]))
        flags = int(rng.choice([0, 0, E.FLAG_SMALL_LISTS, E.FLAG_GENERAL_ONLY, E.FLAG_THETA_WRAP]))
        if flags == E.FLAG_THETA_WRAP and n_theta < 3:
            flags = 0
        d = E.Desc(n_theta, n_rho, -256.0, 256.0, 256.0, 6, -1, T, float(rng.choice([0.0, 4.0, 64.0])), K, dt, n_events, n_hits, max_hpe,
                   flags, 0, 0.0, 0.0)
        h = vp()
        rc = L.hough_plan_create(ctypes.byref(d), ctypes.byref(h))
        if rc != 0:
            continue
        u = rng.uniform(-300, 300, n_hits).astype(np.float32)
        v = rng.uniform(-300, 300, n_hits).astype(np.float32)
        if n_hits > 3:
            u[int(rng.integers(0, n_hits))] = np.nan
            v[int(rng.integers(0, n_hits))] = np.inf
        off = garbage_offsets(rng, n_events, n_hits)
        print(f"case {case}: grid {n_theta}x{n_rho} K {K} events {n_events} hits {n_hits} max_hpe {max_hpe} flags {flags} offsets {off.tolist()}", flush=True)
        du, dv, do = E.DevBuf(u), E.DevBuf(v), E.DevBuf(off)
        cands = E.DevBuf(rng.integers(-2 ** 31, 2 ** 31 - 1, (n_events, K, 8)).astype(np.int32))     # garbage records
        nf = E.DevBuf(garbage_i32(rng, n_events, -3, K + 3))
        labels = E.DevBuf(garbage_i32(rng, max(n_hits, 1), -2, K + 2))
        fits = E.DevBuf(np.zeros((n_events, K), E.FIT_DTYPE))
        geom = E.PlaneGeometry(float(rng.choice([-94.0, 0.0])), float(rng.choice([4.0, 0.25])), int(rng.choice([1, 48, 64])), 5, int(rng.random() < 0.5), 0)
        calls = []
        calls.append(("assign(garbage records)", L.hough_assign_hits(h, du.ptr, dv.ptr, do.ptr, n_events, cands.ptr, nf.ptr, labels.ptr, None)))
        labels2 = E.DevBuf(garbage_i32(rng, max(n_hits, 1), -2, K + 2))
        calls.append(("refit(garbage labels)", L.hough_refit_tracks(h, du.ptr, dv.ptr, do.ptr, n_events, nf.ptr, labels2.ptr, ctypes.byref(geom), fits.ptr, None)))
        calls.append(("find", L.hough_find_clusters(h, du.ptr, dv.ptr, do.ptr, n_events, cands.ptr, nf.ptr, None)))
        calls.append(("assign", L.hough_assign_hits(h, du.ptr, dv.ptr, do.ptr, n_events, cands.ptr, nf.ptr, labels.ptr, None)))
        calls.append(("refit", L.hough_refit_tracks(h, du.ptr, dv.ptr, do.ptr, n_events, nf.ptr, labels.ptr, ctypes.byref(geom), fits.ptr, None)))
        dig = E.DevBuf(np.zeros(n_events, np.uint64))
        calls.append(("vote", L.hough_vote(h, du.ptr, dv.ptr, do.ptr, n_events, None, dig.ptr, None)))
        calls.append(("peeloff", L.hough_find_tracks_peeloff(h, du.ptr, dv.ptr, do.ptr, n_events, cands.ptr, nf.ptr, labels.ptr, None)))
        calls.append(("two_stage", L.hough_find_two_stage(h, du.ptr, dv.ptr, do.ptr, n_events, int(rng.choice([1, 2, 4])), int(rng.choice([1, 4, 8])),
                                                          cands.ptr, nf.ptr, None)))
        # the host-buffer pipeline with the same garbage offsets (its own checks come first: offsets[0] must be 0, the total inside the plan)
        hc, hn, hl = np.zeros((n_events, K), E.CAND_DTYPE), np.zeros(n_events, np.int32), np.zeros(max(n_hits, 1), np.int32)
        calls.append(("run_host", L.hough_run_host_chunked(h, u.ctypes.data, v.ctypes.data, off.ctypes.data, n_events, hc.ctypes.data,
                                                           hn.ctypes.data, hl.ctypes.data, int(rng.choice([0, 1, 3])))))
        dbg = np.zeros(16, np.uint64)
        L.hough_plan_debug_counters(h, dbg.ctypes.data, None)
        L.hough_plan_destroy(h)
        # front end: garbage fill offsets over honest hit arrays
        n_fills = int(rng.integers(1, 5))
        fo = garbage_offsets(rng, n_fills, n_hits)
        wpf = int(rng.integers(1, 12))
        fd = E.FrontDesc(0.0, 10.0, 5.0, wpf, 300.0, n_fills, n_hits, 0, 0)
        fh = vp()
        if L.hough_frontend_create(ctypes.byref(fd), ctypes.byref(fh)) == 0:
            t = rng.uniform(-20, 80, n_hits).astype(np.float32)
            cap = int(rng.choice([0, 1, 2 * n_hits, n_hits // 2 + 1]))
            bx, by, bz, bt, bf = E.DevBuf(u), E.DevBuf(v), E.DevBuf(u), E.DevBuf(t), E.DevBuf(fo)
            bu, bv, bs = E.DevBuf(np.zeros(max(cap, 1), np.float32)), E.DevBuf(np.zeros(max(cap, 1), np.float32)), E.DevBuf(np.zeros(max(cap, 1), np.int32))
            bo = E.DevBuf(np.zeros(n_fills * wpf + 1, np.int64))
            print(f"        front end: fills {fo.tolist()} windows {wpf} capacity {cap}", flush=True)
            calls.append(("frontend", L.hough_frontend_slice(fh, bx.ptr, by.ptr, bz.ptr, bt.ptr, bf.ptr, n_fills, n_hits, bu.ptr, bv.ptr, bs.ptr,
                                                             bo.ptr, cap, None)))
            L.hough_frontend_destroy(fh)
        for name, rc in calls:
            rcs[(name, rc)] = rcs.get((name, rc), 0) + 1
        viol = int(L.cuda_emu_violations())
        if viol or int(dbg[14]):
            bad += 1
            print(f"VIOLATION in case {case}: model {viol} ({L.cuda_emu_first_violation().decode()}), index checks {int(dbg[14])} first at site {int(dbg[13])}", flush=True)
    print(f"fuzz_hostile seed {a.seed}: {a.cases} cases, {bad} with a violation; return codes: "
          + ", ".join(f"{n} -> {rc}: {c}" for (n, rc), c in sorted(rcs.items())))
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
