"""GPU parity of the stages around the Hough core (front end: time slicing + phi; back end: line refit + found criterion)
against oracle/track_def.py, through the C ABI.  Integer outputs and the fp32 values are compared bit for bit (both sides run
the same integer algorithm; the fp32 parameters only need 1e-5 relative, BASELINE.json north_star)."""
import numpy as np
import pytest
import torch

from oracle import hough_c as C
from oracle import hough_def as D
from oracle import track_def as T
from paper_2511_02742_b200 import hough as H
from paper_2511_02742_b200 import synth
from util import fills_with_tracks, params_of, synthetic_fills

pytestmark = pytest.mark.gpu

GEOM = T.PlaneGeometry(origin=-94.0, pitch=4.0, n_planes=48)


def dev(a, dt):
    return torch.from_numpy(np.ascontiguousarray(a, dt)).cuda()


def gpu_slice(fe, x, y, z, t, fo, capacity=None):
    h = H.hough_frontend_create(fe.t0, fe.width, fe.step, fe.windows_per_fill, max(1, len(fo) - 1), len(x), fe.xy_max)
    u, v, src, off = H.hough_frontend_slice(h, dev(x, np.float32), dev(y, np.float32), dev(z, np.float32), dev(t, np.float32),
                                            dev(fo, np.int64), capacity)
    torch.cuda.synchronize()
    st = H.hough_frontend_status(h)
    H.hough_frontend_destroy(h)
    return u, v, src, off, st


def gpu_refit(p, u, v, offsets, n_found, labels, geom, dt=H.HOUGH_I32):
    E = len(offsets) - 1
    plan = H.hough_plan_create(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window,
                               p.max_candidates, max(1, E), len(u), max(1, int(np.diff(offsets).max())), dt, p.hit_frac_bits, p.acc_frac_bits)
    fits = H.hough_refit_tracks(plan, dev(u, np.float32), dev(v, np.float32), dev(offsets, np.int64), dev(n_found, np.int32),
                                dev(labels, np.int32), geom.origin, geom.pitch, geom.n_planes, geom.min_run, geom.wrap)
    torch.cuda.synchronize()
    dbg = H.hough_plan_debug_counters(plan)
    assert int(dbg[14]) == 0
    H.hough_plan_destroy(plan)
    return H.fits_to_numpy(fits)


def fits_equal(row, oracle_fits):
    for s, f in enumerate(oracle_fits):
        g = row[s]
        assert (int(g["n_hits"]), int(g["plane_mask"]), int(g["max_run"]), int(g["flags"]), int(g["reserved"])) == \
               (f.n_hits, f.plane_mask, f.max_run, f.flags, 0), (s, g, f)
        np.testing.assert_allclose(g["slope"], f.slope, rtol=1e-5, atol=0)
        np.testing.assert_allclose(g["intercept"], f.intercept, rtol=1e-5, atol=0)
        assert g["slope"].tobytes() == f.slope.tobytes() and g["intercept"].tobytes() == f.intercept.tobytes()


@pytest.mark.gate
@pytest.mark.parametrize("fe", [T.FrontEnd(windows_per_fill=12), T.FrontEnd(t0=-3.5, width=10.0, step=2.5, windows_per_fill=20),
                                T.FrontEnd(t0=1.0, width=4.0, step=6.0, windows_per_fill=7)],
                         ids=["10ns_5ns", "four_fold_overlap", "gaps_between_windows"])
def test_frontend_slice(fe):
    x, y, z, t, fo = synthetic_fills(40, seed=41, hits_per_fill=3000)
    ou, ov, osrc, ooff = T.slice_batch(x, y, z, t, fo, fe)
    u, v, src, off, st = gpu_slice(fe, x, y, z, t, fo)
    assert st == 0
    np.testing.assert_array_equal(off.cpu().numpy(), ooff)
    M = int(ooff[-1])
    np.testing.assert_array_equal(src[:M].cpu().numpy(), osrc)
    assert u[:M].cpu().numpy().tobytes() == ou.tobytes() and v[:M].cpu().numpy().tobytes() == ov.tobytes()


def test_frontend_one_large_fill_and_truncation():
    fe = T.FrontEnd(windows_per_fill=200)
    x, y, z, t, fo = synthetic_fills(1, seed=44, hits_per_fill=60000, t_span=1000.0)
    _, _, osrc, ooff = T.slice_batch(x, y, z, t, fo, fe)
    u, v, src, off, st = gpu_slice(fe, x, y, z, t, fo)
    assert st == 0
    np.testing.assert_array_equal(off.cpu().numpy(), ooff)
    np.testing.assert_array_equal(src[: int(ooff[-1])].cpu().numpy(), osrc)
    cap = int(ooff[-1]) // 3
    u, v, src, off, st = gpu_slice(fe, x, y, z, t, fo, capacity=cap)
    assert st & H.HOUGH_STATUS_OUTPUT_TRUNCATED
    np.testing.assert_array_equal(off.cpu().numpy(), ooff)
    np.testing.assert_array_equal(src[:cap].cpu().numpy(), osrc[:cap])


@pytest.mark.gate
@pytest.mark.parametrize("cfg,n_events,geom", [(1, 8, GEOM), (3, 3, GEOM)])
def test_refit_gate(cfg, n_events, geom):
    check_refit(cfg, n_events, geom)


@pytest.mark.parametrize("cfg,n_events,geom", [(1, 1500, GEOM), (3, 300, GEOM), (2, 400, T.PlaneGeometry(-94.0, 4.0, 48, min_run=7, wrap=True))])
def test_refit_tracks(cfg, n_events, geom):
    check_refit(cfg, n_events, geom)


def check_refit(cfg, n_events, geom):
    wl = synth.workload(cfg)
    wl = wl.with_events(max(wl.n_events, n_events))
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    o = C.run_batch(b.u, b.v, b.offsets, p)
    fits = gpu_refit(p, b.u, b.v, b.offsets, o["n_found"], o["labels"], geom, H.HOUGH_U16 if wl.count_dtype == "u16" else H.HOUGH_I32)
    step = max(1, n_events // 40)                      # the Python oracle checks a sample of the events, every record of each
    for e in range(0, n_events, step):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        nk = min(int(o["n_found"][e]), p.max_candidates)
        fits_equal(fits[e], T.refit_event(b.u[a:z], b.v[a:z], o["labels"][a:z], nk, p, geom))
        assert (fits[e, nk:]["n_hits"] == 0).all()


def test_frontend_skips_fills_whose_range_is_not_inside_the_hits():
    """Fill offsets are caller data: a fill that ends beyond n_hits, starts below 0 or ends before it starts is skipped and flagged."""
    fe = T.FrontEnd(windows_per_fill=6)
    x, y, z, t, fo = synthetic_fills(4, seed=44)
    n = len(x)
    for bad in ([0, int(fo[1]), n + 100, int(fo[3]), n], [0, -5, int(fo[2]), int(fo[3]), n], [0, int(fo[2]), int(fo[1]), int(fo[3]), 2 ** 40]):
        assert gpu_slice(fe, x, y, z, t, np.array(bad, np.int64))[4] & H.HOUGH_STATUS_BAD_OFFSETS
    assert gpu_slice(fe, x, y, z, t, fo)[4] == 0


def test_refit_ignores_labels_beyond_the_kept_records():
    """Labels are caller data: one that names no kept record of its event must not index the per-candidate sums."""
    from test_emulated_kernels import fits_equal, GEOM
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 5)
    p = params_of(wl)
    o = C.run_batch(b.u, b.v, b.offsets, p)
    labels = o["labels"].copy()
    labels[::7] = np.array([p.max_candidates, p.max_candidates + 1, 99, 130], np.int32)[np.arange(len(labels[::7])) % 4]
    plan = H.hough_plan_create(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window,
                               p.max_candidates, 5, len(b.u), int(np.diff(b.offsets).max()))
    fits = H.fits_to_numpy(H.hough_refit_tracks(plan, torch.from_numpy(b.u).cuda(), torch.from_numpy(b.v).cuda(),
                                                torch.from_numpy(b.offsets).cuda(), torch.from_numpy(o["n_found"]).cuda(),
                                                torch.from_numpy(labels).cuda(), GEOM.origin, GEOM.pitch, GEOM.n_planes))
    H.hough_plan_destroy(plan)
    for e in range(5):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        nk = min(int(o["n_found"][e]), p.max_candidates)
        lab = labels[a:z].copy()
        lab[lab >= nk] = -1
        fits_equal(fits[e], T.refit_event(b.u[a:z], b.v[a:z], lab, nk, p, GEOM))


def test_refit_rejects_plans_whose_sums_could_overflow():
    plan = H.hough_plan_create(64, 512, -1415.0, 1415.0, 1000.0, 3, 6.0, 16, 1, 4, 4)
    z4 = torch.zeros(4, device="cuda")
    with pytest.raises(H.HoughError) as ei:
        H.hough_refit_tracks(plan, z4, z4, torch.tensor([0, 4], device="cuda"), torch.zeros(1, dtype=torch.int32, device="cuda"),
                             torch.full((4,), -1, dtype=torch.int32, device="cuda"), -94.0, 4.0, 48)
    assert ei.value.status == H.HOUGH_ERANGE
    H.hough_plan_destroy(plan)


def test_whole_chain_fills_to_fits():
    """Fills -> windows (front end) -> vote / clusters / assign -> refit, all on the device, each stage against its oracle."""
    fe = T.FrontEnd(windows_per_fill=6)
    x, y, z, t, fo = fills_with_tracks(60, seed=43)
    ou, ov, osrc, ooff = T.slice_batch(x, y, z, t, fo, fe)
    u, v, src, off, st = gpu_slice(fe, x, y, z, t, fo)
    M = int(ooff[-1])
    assert st == 0 and u[:M].cpu().numpy().tobytes() == ou.tobytes()
    p = D.Params(180, 1000, -500.0, 500.0, 256.0, 12, 2.0, 8)               # the paper's grid
    E = len(ooff) - 1
    plan = H.hough_plan_create(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window,
                               p.max_candidates, E, M, max(1, int(np.diff(ooff).max())))
    du, dv = u[:M].contiguous(), v[:M].contiguous()
    cands, n_found = H.hough_find_clusters(plan, du, dv, off)
    labels = H.hough_assign_hits(plan, du, dv, off, cands, n_found)
    fits = H.hough_refit_tracks(plan, du, dv, off, n_found, labels, -175.5, 9.0, 40, 5, True)
    torch.cuda.synchronize()
    o = C.run_batch(ou, ov, ooff, p)
    np.testing.assert_array_equal(n_found.cpu().numpy(), o["n_found"])
    np.testing.assert_array_equal(labels.cpu().numpy(), o["labels"])
    vanes40 = T.PlaneGeometry(origin=-175.5, pitch=9.0, n_planes=40, min_run=5, wrap=True)
    fn = H.fits_to_numpy(fits)
    found = 0
    for e in range(E):
        a, zz = int(ooff[e]), int(ooff[e + 1])
        nk = min(int(o["n_found"][e]), p.max_candidates)
        fo_e = T.refit_event(ou[a:zz], ov[a:zz], o["labels"][a:zz], nk, p, vanes40)
        fits_equal(fn[e], fo_e)
        found += sum(1 for f in fo_e if f.flags & T.FIT_FOUND)
    assert found >= 60
    H.hough_plan_destroy(plan)


@pytest.mark.parametrize("grid,K,w_bins", [((64, 128), 8, 1.5), ((180, 1000), 6, 2.0)])
def test_peeloff_variant(grid, K, w_bins):
    """O13 on the GPU against the step-by-step oracle: tracks in the order found, labels."""
    from test_emulated_kernels import peel_case
    p = D.Params(grid[0], grid[1], -256.0, 256.0, 256.0, 12, w_bins * 512.0 / grid[1], K)
    us, vs, offs = [], [], [0]
    for e, (nt, nn) in enumerate([(3, 12), (0, 0), (1, 40), (4, 5), (0, 25), (2, 0)] * 3):
        u, v = peel_case(70 + e, nt, nn) if nt + nn else (np.zeros(0, np.float32), np.zeros(0, np.float32))
        us.append(u); vs.append(v); offs.append(offs[-1] + len(u))
    u, v, offsets = np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)
    E = len(offsets) - 1
    plan = H.hough_plan_create(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window,
                               p.max_candidates, E, len(u), int(np.diff(offsets).max()))
    cands, n_found, labels = H.hough_find_tracks_peeloff(plan, dev(u, np.float32), dev(v, np.float32), dev(offsets, np.int64))
    torch.cuda.synchronize()
    assert H.hough_plan_status(plan) == 0 and int(H.hough_plan_debug_counters(plan)[14]) == 0
    gc, gn, gl = H.candidates_to_numpy(cands), n_found.cpu().numpy(), labels.cpu().numpy()
    H.hough_plan_destroy(plan)
    for e in range(E):
        a, z = int(offsets[e]), int(offsets[e + 1])
        tracks, lab = T.peel_event(u[a:z], v[a:z], p)
        assert int(gn[e]) == len(tracks)
        assert [(int(c["theta_bin"]), int(c["rho_bin"]), int(c["votes"])) for c in gc[e, :len(tracks)]] == tracks
        np.testing.assert_array_equal(gl[a:z], lab)


@pytest.mark.parametrize("grid,factors,K", [((180, 256), (4, 4), 16), ((180, 1000), (4, 8), 8)])
def test_two_stage_variant(grid, factors, K):
    """O14 on the GPU against the step-by-step oracle: ranked candidates with their exact counts."""
    from test_emulated_kernels import peel_case
    p = D.Params(grid[0], grid[1], -256.0, 256.0, 256.0, 12, 512.0 / grid[1], K)
    us, vs, offs = [], [], [0]
    for e, (nt, nn) in enumerate([(3, 12), (0, 0), (1, 40), (5, 30), (0, 25), (2, 3)] * 4):
        u, v = peel_case(80 + e, nt, nn) if nt + nn else (np.zeros(0, np.float32), np.zeros(0, np.float32))
        us.append(u); vs.append(v); offs.append(offs[-1] + len(u))
    u, v, offsets = np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)
    E = len(offsets) - 1
    plan = H.hough_plan_create(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window,
                               p.max_candidates, E, len(u), int(np.diff(offsets).max()))
    cands, n_found = H.hough_find_two_stage(plan, dev(u, np.float32), dev(v, np.float32), dev(offsets, np.int64), *factors)
    torch.cuda.synchronize()
    assert H.hough_plan_status(plan) == 0 and int(H.hough_plan_debug_counters(plan)[14]) == 0
    gc, gn = H.candidates_to_numpy(cands), n_found.cpu().numpy()
    H.hough_plan_destroy(plan)
    for e in range(E):
        a, z = int(offsets[e]), int(offsets[e + 1])
        want, n = T.two_stage_event(u[a:z], v[a:z], p, *factors)
        assert int(gn[e]) == n
        assert [(int(c["theta_bin"]), int(c["rho_bin"]), int(c["votes"])) for c in gc[e, :n]] == want
