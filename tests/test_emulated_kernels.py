"""The CUDA kernels of paper_2511_02742_b200/csrc, compiled for the host execution model of tests/emu/cuda_emu.h, against the
CPU oracle -- element by element, through the same C ABI, on a machine WITHOUT a GPU.

What this proves: the kernels' logic (index arithmetic, list capacities and the hand-over to the general kernel, barrier
placement against the data flow, per-event resets when one CTA processes many events, results independent of the thread
schedule) with every shared-memory and "device"-memory access bounds-checked -- the kernels' own -DHOUGH_BOUNDS checks are
compiled in, shared-window addresses of the PTX accesses are validated, and every allocation ends at an inaccessible page.
What it does not prove: anything about the hardware (memory model, PTX semantics, timing).  The GPU parity tests
(tests/test_gpu_parity.py, -m gpu) are the proof of record; these cases mirror them at sizes the model runs in seconds.
"""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "emu"))
import hough_emu as E  # noqa: E402

from oracle import hough_c as C  # noqa: E402
from oracle import hough_def as D  # noqa: E402
from paper_2511_02742_b200 import synth  # noqa: E402
from test_oracle_pins import edge_cases  # noqa: E402
from util import fills_with_tracks, mixed_batch, paper_grid_batch, params_of, std_params, synthetic_fills  # noqa: E402

INT_FIELDS = ("theta_bin", "rho_bin", "votes", "cluster_root", "cluster_nbins", "reserved")


@pytest.fixture(autouse=True)
def default_schedule():
    E.configure(seed=1, preempt_per_1024=0, smem_window=1024)
    yield
    E.configure(seed=1, preempt_per_1024=0, smem_window=1024)


def assert_same(g, o, p, status=0):
    assert g["emu_violations"] == 0, g["emu_first_violation"]
    assert g["bounds_violations"] == 0, f"index check failed inside a kernel, first at site {g['bounds_site']}"
    assert g["status"] == status
    if "acc" in g and o.get("acc") is not None:
        np.testing.assert_array_equal(g["acc"], o["acc"])
    if "digest" in g:
        np.testing.assert_array_equal(g["digest"], o["digest"])
    np.testing.assert_array_equal(g["n_found"], o["n_found"])
    for e in range(len(o["n_found"])):
        k = min(int(o["n_found"][e]), p.max_candidates)
        ge, oe = g["cands"][e, :k], o["cands"][e, :k]
        for f in INT_FIELDS:
            np.testing.assert_array_equal(ge[f], oe[f], err_msg=f"event {e} field {f}")
        np.testing.assert_allclose(ge["theta"], oe["theta"], rtol=1e-5, atol=0)
        np.testing.assert_allclose(ge["rho"], oe["rho"], rtol=1e-5, atol=0)
    np.testing.assert_array_equal(g["labels"], o["labels"])


def oracle_run(p, u, v, offsets, want_acc=True):
    return C.run_batch(u, v, offsets, p, want_digest=True, want_acc=want_acc)


def dtype_of(wl):
    return E.HOUGH_U16 if wl.count_dtype == "u16" else E.HOUGH_I32


# ----------------------------------------------------------------------------- BASELINE configs
@pytest.mark.parametrize("cfg,n_events", [(0, 1), (1, 40), (2, 12), (3, 6)])
@pytest.mark.parametrize("flags", [0, E.FLAG_SMALL_LISTS, E.FLAG_GENERAL_ONLY], ids=["fast", "small_lists", "general_only"])
def test_configs_bit_exact(cfg, n_events, flags):
    wl = synth.workload(cfg)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    g = E.run(p, b.u, b.v, b.offsets, dtype_of(wl), flags=flags)
    o = oracle_run(p, b.u, b.v, b.offsets)
    assert_same(g, o, p)
    if flags == 0:
        assert g["info"]["fast_groups"] > 0 and g["deferred"] == 0       # S1-S4 ran in the fast kernel
    elif flags == E.FLAG_GENERAL_ONLY:
        assert g["info"]["fast_groups"] == 0 and g["deferred"] == 0
    elif cfg in (1, 3):
        assert g["deferred"] > 0                                           # the lists overflowed: handed to the general kernel


@pytest.mark.parametrize("seed,preempt", [(2, 0), (3, 8), (4, 64), (5, 512)])
def test_results_do_not_depend_on_the_schedule(seed, preempt):
    """Other fiber orders, and a thread switch with probability preempt/1024 at every atomic / cache-bypassing access: lists are
    filled in another order, union-find races resolve differently -- the outputs may not change."""
    E.configure(seed=seed, preempt_per_1024=preempt)
    wl = synth.workload(3)
    b = synth.generate(wl, 3, 2)
    p = params_of(wl)
    for flags in (0, E.FLAG_GENERAL_ONLY):
        g = E.run(p, b.u, b.v, b.offsets, E.HOUGH_U16, flags=flags, want_vote=False)
        o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
        assert_same(g, o, p)


@pytest.mark.parametrize("window", [0, 1024, 3840, 4096, 8192 + 128])
def test_shared_window_offset(window):
    """The vote of the fast kernel folds the tile's shared-window address into the fixed-point offset; the host sized that
    for a tile below 4096.  Elsewhere the kernel must notice and leave every event to the general kernel."""
    E.configure(seed=1, smem_window=window)
    wl = synth.workload(3)
    b = synth.generate(wl, 0, 2)
    p = params_of(wl)
    g = E.run(p, b.u, b.v, b.offsets, E.HOUGH_U16, want_vote=False)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    assert_same(g, o, p)
    assert g["deferred"] == (0 if window < 4096 and window % 256 == 0 else 2)


@pytest.mark.parametrize("workers,flags", [(4, 0), (6, E.FLAG_SMALL_LISTS), (5, E.FLAG_GENERAL_ONLY)])
def test_concurrent_ctas(workers, flags):
    """Several persistent CTAs at the same time, each on its own OS thread: they share the work counter, the deferred list and
    the status word through real atomics, and each uses its own slab of the general kernel's global scratch (blockIdx > 0)."""
    E.configure(seed=7, workers=workers)
    try:
        wl, u, v, offsets, kinds = mixed_batch(3, 48, seed=29)
        p = params_of(wl)
        g = E.run(p, u, v, offsets, E.HOUGH_U16, flags=flags, want_acc=False)
        o = oracle_run(p, u, v, offsets, want_acc=False)
        assert_same(g, o, p)
        if flags == 0:
            assert g["deferred"] == kinds.count("count>1023")
    finally:
        E.configure(seed=1, workers=1)


def test_many_events_per_cta():
    """The model runs the CTAs of a grid one after another, so the first CTA of the persistent grid processes EVERY event:
    per-event resets (halos, lists, histogram, control block), tile reuse across events, the work counter."""
    wl = synth.workload(3)
    b = synth.generate(wl, 0, 24)
    p = params_of(wl)
    g = E.run(p, b.u, b.v, b.offsets, E.HOUGH_U16, want_acc=False)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    assert_same(g, o, p)
    assert g["info"]["fast_groups"] > 0 and g["deferred"] == 0


def test_mixed_batch_with_deferred_events_interleaved():
    wl, u, v, offsets, kinds = mixed_batch(1, 400, seed=21)
    p = params_of(wl)
    n_big = kinds.count("count>1023")
    assert n_big >= 3 and kinds.count("empty") >= 5 and kinds.count("invalid") >= 1
    g = E.run(p, u, v, offsets, max_hpe=2048, want_acc=False)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert_same(g, o, p)
    assert g["info"]["fast_groups"] > 0 and g["deferred"] == n_big


def test_events_longer_than_the_fast_staging_buffer_are_deferred():
    wl, u, v, offsets, kinds = mixed_batch(2, 60, seed=23, long_hits=9000)
    p = params_of(wl)
    n_long = kinds.count("long")
    assert n_long >= 1
    g = E.run(p, u, v, offsets, max_hpe=9000, want_acc=False)
    assert g["info"]["fast_hits_cap"] < 9000
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert_same(g, o, p)
    assert g["deferred"] == n_long + kinds.count("count>1023")


@pytest.mark.parametrize("hits_idx", [0, 1, 2, 3])
@pytest.mark.parametrize("grid_idx", [0, 1, 2, 3])
def test_config4_cells(hits_idx, grid_idx):
    wl = synth.workload(4, hits_idx, grid_idx)
    n_events = {0: 12, 1: 8, 2: 3, 3: 2}[hits_idx]
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    g = E.run(p, b.u, b.v, b.offsets, want_acc=grid_idx < 3)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=grid_idx < 3)
    assert_same(g, o, p)


# ----------------------------------------------------------------------------- adversarial edge set
@pytest.mark.parametrize("case", edge_cases(), ids=lambda c: c[0])
def test_edge_set(case):
    name, p, u, v = case
    offsets = np.array([0, len(u)], np.int64)
    for flags in (0, E.FLAG_GENERAL_ONLY):
        g = E.run(p, u, v, offsets, max_hpe=max(len(u), 1), flags=flags)
        o = oracle_run(p, u, v, offsets)
        assert_same(g, o, p)


def test_edge_set_as_one_ragged_batch():
    cases = [c for c in edge_cases() if c[1] == edge_cases()[0][1]]
    p = cases[0][1]
    us, vs, offs = [], [], [0]
    for _, _, u, v in cases:
        us.append(u); vs.append(v); offs.append(offs[-1] + len(u)); offs.append(offs[-1])
    u, v, offsets = np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)
    g = E.run(p, u, v, offsets)
    o = oracle_run(p, u, v, offsets)
    assert_same(g, o, p)


def test_strip_seams_dense_mask():
    rng = np.random.default_rng(12)
    p = std_params(512, 512, T=3, K=128)
    u = rng.uniform(-94, 94, 1500).astype(np.float32)
    v = rng.uniform(-194, 194, 1500).astype(np.float32)
    offsets = np.array([0, 700, 1500], np.int64)
    for flags in (0, E.FLAG_GENERAL_ONLY):
        g = E.run(p, u, v, offsets, flags=flags)
        o = oracle_run(p, u, v, offsets)
        assert_same(g, o, p)


def test_ties_at_the_kth_vote_count():
    """More peaks than K with many ties at the K-th count: the tie path of the fast kernel's selection (the count
    of kept peaks was overwritten while other warps still read it)."""
    rng = np.random.default_rng(14)
    p = std_params(256, 256, T=3, K=24)
    u = rng.uniform(-94, 94, 260).astype(np.float32)
    v = rng.uniform(-194, 194, 260).astype(np.float32)
    offsets = np.array([0, 130, 260], np.int64)
    for seed in (1, 2, 3):
        E.configure(seed=seed, preempt_per_1024=32)
        g = E.run(p, u, v, offsets)
        o = oracle_run(p, u, v, offsets)
        assert (o["n_found"] > p.max_candidates).all()
        assert_same(g, o, p)
        assert g["info"]["fast_groups"] > 0 and g["deferred"] == 0


def test_unsafe_hits_near_the_rho_range_edge():
    rng = np.random.default_rng(11)
    p = std_params(256, 256, T=4, K=64)
    u = rng.uniform(-256, 256, 600).astype(np.float32)
    v = rng.uniform(-256, 256, 600).astype(np.float32)
    offsets = np.array([0, 100, 100, 350, 600], np.int64)
    g = E.run(p, u, v, offsets)
    o = oracle_run(p, u, v, offsets)
    assert_same(g, o, p)
    assert g["acc"].sum() < 600 * 256


def test_large_K_and_overflowing_peak_list():
    rng = np.random.default_rng(13)
    p = std_params(512, 512, T=1, K=4096)
    u = rng.uniform(-94, 94, 300).astype(np.float32)
    v = rng.uniform(-194, 194, 300).astype(np.float32)
    offsets = np.array([0, 300], np.int64)
    g = E.run(p, u, v, offsets, want_acc=False)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert o["n_found"][0] > 4096
    assert_same(g, o, p)


def test_many_hits_per_event_is_staged_in_chunks():
    wl = synth.workload(4, 3, 1)
    b = synth.generate(wl, 0, 2)
    p = params_of(wl, max_candidates=16)
    g = E.run(p, b.u, b.v, b.offsets, flags=E.FLAG_GENERAL_ONLY)
    o = oracle_run(p, b.u, b.v, b.offsets)
    assert_same(g, o, p)


def test_status_word_flags_long_events():
    p = std_params(64, 64, T=3, K=8)
    rng = np.random.default_rng(2)
    u = rng.uniform(-100, 100, 300).astype(np.float32)
    v = rng.uniform(-100, 100, 300).astype(np.float32)
    offsets = np.array([0, 50, 250, 300], np.int64)
    g = E.run(p, u, v, offsets, max_hpe=100, want_vote=False)
    assert g["emu_violations"] == 0 and g["bounds_violations"] == 0
    assert g["status"] & 1
    assert g["n_found"][1] == 0 and (g["labels"][50:250] == -1).all()
    o = C.run_batch(u[:50], v[:50], np.array([0, 50], np.int64), p)
    np.testing.assert_array_equal(g["labels"][:50], o["labels"])


def test_paper_grid_180x1000_multi_event():
    p, u, v, offsets = paper_grid_batch(24)
    g = E.run(p, u, v, offsets, want_acc=False)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert_same(g, o, p)


@pytest.mark.parametrize("n_chunks,n_events", [(0, 12), (3, 40), (7, 40), (32, 40)])
def test_run_host_chunked(n_chunks, n_events):
    wl = synth.workload(1)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    offsets = np.concatenate([b.offsets[:n_events // 2], np.repeat(b.offsets[n_events // 2], 3), b.offsets[n_events // 2:]])
    g = E.run_host(p, b.u, b.v, offsets, n_chunks, repeat=2)
    assert g["emu_violations"] == 0, g["emu_first_violation"]
    o = C.run_batch(b.u, b.v, offsets, p)
    np.testing.assert_array_equal(g["n_found"], o["n_found"])
    np.testing.assert_array_equal(g["labels"], o["labels"])
    for e in range(len(offsets) - 1):
        k = min(int(o["n_found"][e]), p.max_candidates)
        assert g["cands"][e, :k].tobytes() == o["cands"][e, :k].tobytes()


# ----------------------------------------------------------------------------- stages around the core (O9-O12)
from oracle import track_def as T  # noqa: E402

GEOM = T.PlaneGeometry(origin=-94.0, pitch=4.0, n_planes=48)


def fits_equal(fits_row, oracle_fits):
    for s, f in enumerate(oracle_fits):
        g = fits_row[s]
        assert (int(g["n_hits"]), int(g["plane_mask"]), int(g["max_run"]), int(g["flags"]), int(g["reserved"])) == \
               (f.n_hits, f.plane_mask, f.max_run, f.flags, 0), (s, g, f)
        assert g["slope"].tobytes() == f.slope.tobytes() and g["intercept"].tobytes() == f.intercept.tobytes(), (s, g, f)


@pytest.mark.parametrize("cfg,n_events,geom", [(1, 12, GEOM), (3, 3, GEOM), (2, 5, T.PlaneGeometry(-94.0, 4.0, 48, min_run=7, wrap=True))])
def test_refit_tracks(cfg, n_events, geom):
    """O9 + O10: per kept candidate the exact integer sums, plane mask, longest run and the line, bit for bit."""
    wl = synth.workload(cfg)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    o = C.run_batch(b.u, b.v, b.offsets, p)
    fits, rc = E.refit(p, b.u, b.v, b.offsets, o["n_found"], o["labels"], geom, dtype_of(wl))
    assert rc == 0
    for e in range(n_events):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        nk = min(int(o["n_found"][e]), p.max_candidates)
        fits_equal(fits[e], T.refit_event(b.u[a:z], b.v[a:z], o["labels"][a:z], nk, p, geom))
        assert (fits[e, nk:]["n_hits"] == 0).all()                       # rows beyond n_kept are untouched


def test_refit_rejects_plans_whose_sums_could_overflow():
    p = D.Params(64, 512, -1415.0, 1415.0, 1000.0, 3, 6.0, 16, 6, -1)    # coord_max 2^H = 64000 > 2^15
    u = np.zeros(4, np.float32)
    _, rc = E.refit(p, u, u, np.array([0, 4], np.int64), np.zeros(1, np.int32), np.full(4, -1, np.int32), GEOM)
    assert rc == -2


@pytest.mark.parametrize("fe", [T.FrontEnd(windows_per_fill=12), T.FrontEnd(t0=-3.5, width=10.0, step=2.5, windows_per_fill=20),
                                T.FrontEnd(t0=1.0, width=4.0, step=6.0, windows_per_fill=7)],
                         ids=["10ns_5ns", "four_fold_overlap", "gaps_between_windows"])
def test_frontend_slice(fe):
    """O11 + O12: window membership, input order inside a window, CORDIC phi and the event offsets, bit for bit."""
    x, y, z, t, fo = synthetic_fills(5, seed=41)
    ou, ov, osrc, ooff = T.slice_batch(x, y, z, t, fo, fe)
    g = E.frontend_slice(fe, x, y, z, t, fo)
    assert g["status"] == 0
    np.testing.assert_array_equal(g["offsets"], ooff)
    M = int(ooff[-1])
    assert M > 0
    np.testing.assert_array_equal(g["src"][:M], osrc)
    assert g["u"][:M].tobytes() == ou.tobytes() and g["v"][:M].tobytes() == ov.tobytes()
    assert (g["src"][M:] == -1).all()                                       # nothing is written past the last window


def test_frontend_reports_truncation_and_still_writes_all_offsets():
    fe = T.FrontEnd(windows_per_fill=12)
    x, y, z, t, fo = synthetic_fills(3, seed=42)
    _, _, osrc, ooff = T.slice_batch(x, y, z, t, fo, fe)
    cap = int(ooff[-1]) // 2
    g = E.frontend_slice(fe, x, y, z, t, fo, capacity=cap)
    assert g["status"] & 8
    np.testing.assert_array_equal(g["offsets"], ooff)
    np.testing.assert_array_equal(g["src"][:cap], osrc[:cap])


def test_frontend_feeds_the_hough_core():
    """Fills -> windows -> vote / clusters / assign -> refit, every stage against its oracle on the previous stage's output."""
    fe = T.FrontEnd(windows_per_fill=6)
    x, y, z, t, fo = fills_with_tracks(3, seed=43)
    g = E.frontend_slice(fe, x, y, z, t, fo)
    ou, ov, osrc, ooff = T.slice_batch(x, y, z, t, fo, fe)
    M = int(ooff[-1])
    np.testing.assert_array_equal(g["offsets"], ooff)
    assert g["u"][:M].tobytes() == ou.tobytes()
    p = D.Params(180, 1000, -500.0, 500.0, 256.0, 12, 2.0, 8)               # the paper's grid
    h = E.run(p, g["u"][:M], g["v"][:M], g["offsets"], want_acc=False)
    o = oracle_run(p, ou, ov, ooff, want_acc=False)
    assert_same(h, o, p)
    assert (o["n_found"] >= 1).sum() >= 3                                   # the windows that hold a track find it
    vanes40 = T.PlaneGeometry(origin=-175.5, pitch=9.0, n_planes=40, min_run=5, wrap=True)
    fits, rc = E.refit(p, ou, ov, ooff, o["n_found"], o["labels"], vanes40)
    assert rc == 0
    found = 0
    for e in range(len(ooff) - 1):
        a, zz = int(ooff[e]), int(ooff[e + 1])
        nk = min(int(o["n_found"][e]), p.max_candidates)
        fo_e = T.refit_event(ou[a:zz], ov[a:zz], o["labels"][a:zz], nk, p, vanes40)
        fits_equal(fits[e], fo_e)
        found += sum(1 for f in fo_e if f.flags & T.FIT_FOUND)
    assert found >= 3


def peel_case(seed, n_tracks, n_noise):
    rng = np.random.default_rng(seed)
    us, vs = [], []
    for _ in range(n_tracks):
        uu, vv = synth.ideal_track(rng.uniform(-1, 1), rng.uniform(-100, 100))
        keep = rng.random(48) > 0.1
        us.append(uu[keep]); vs.append((vv + rng.normal(0, 0.1, 48).astype(np.float32))[keep])
    us.append(rng.uniform(-94, 94, n_noise).astype(np.float32)); vs.append(rng.uniform(-194, 194, n_noise).astype(np.float32))
    u, v = np.concatenate(us), np.concatenate(vs)
    pm = rng.permutation(len(u))
    return u[pm], v[pm]


@pytest.mark.parametrize("grid,K,w_bins", [((64, 128), 8, 1.5), ((45, 300), 2, 1.0), ((90, 77), 6, 0.25)])
def test_peeloff_variant(grid, K, w_bins):
    """O13: the paper's own peak rule, one track at a time, against the step-by-step oracle (tracks in the order found, labels)."""
    p = std_params(grid[0], grid[1], T=12, K=K, w_bins=w_bins)
    us, vs, offs = [], [], [0]
    for e, (nt, nn) in enumerate([(3, 12), (0, 0), (1, 40), (4, 5), (0, 25)]):
        u, v = peel_case(50 + e, nt, nn) if nt + nn else (np.zeros(0, np.float32), np.zeros(0, np.float32))
        us.append(u); vs.append(v); offs.append(offs[-1] + len(u))
    u, v, offsets = np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)
    u[5] = np.nan                                                           # an invalid hit: never on a track
    g = E.peeloff(p, u, v, offsets)
    assert g["status"] == 0
    for e in range(len(offsets) - 1):
        a, z = int(offsets[e]), int(offsets[e + 1])
        tracks, labels = T.peel_event(u[a:z], v[a:z], p)
        assert int(g["n_found"][e]) == len(tracks)
        got = [(int(c["theta_bin"]), int(c["rho_bin"]), int(c["votes"])) for c in g["cands"][e, :len(tracks)]]
        assert got == tracks
        assert [int(c["cluster_root"]) for c in g["cands"][e, :len(tracks)]] == list(range(len(tracks)))
        np.testing.assert_array_equal(g["labels"][a:z], labels)
    assert g["n_found"][0] >= (2 if w_bins >= 1.0 else 1) and g["labels"][5] == -1


@pytest.mark.parametrize("grid,factors,K", [((180, 256), (4, 4), 16), ((180, 1000), (4, 8), 8), ((64, 64), (1, 1), 16), ((90, 100), (7, 3), 4)])
def test_two_stage_variant(grid, factors, K):
    """O14: the paper's coarse -> fine two-stage histogram against the step-by-step oracle (ranked candidates, counts)."""
    p = D.Params(grid[0], grid[1], -256.0, 256.0, 256.0, 12, 512.0 / grid[1], K)
    us, vs, offs = [], [], [0]
    for e, (nt, nn) in enumerate([(3, 12), (0, 0), (1, 40), (5, 30), (0, 25)]):
        u, v = peel_case(60 + e, nt, nn) if nt + nn else (np.zeros(0, np.float32), np.zeros(0, np.float32))
        us.append(u); vs.append(v); offs.append(offs[-1] + len(u))
    u, v, offsets = np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)
    g = E.two_stage(p, u, v, offsets, *factors)
    assert g["rc"] == 0
    total = 0
    for e in range(len(offsets) - 1):
        a, z = int(offsets[e]), int(offsets[e + 1])
        want, n = T.two_stage_event(u[a:z], v[a:z], p, *factors)
        assert int(g["n_found"][e]) == n
        got = [(int(c["theta_bin"]), int(c["rho_bin"]), int(c["votes"])) for c in g["cands"][e, :n]]
        assert got == want
        assert [int(c["cluster_root"]) for c in g["cands"][e, :n]] == list(range(n))
        total += n
    assert total >= 4


def test_two_stage_rejects_a_coarse_grid_that_does_not_fit_shared_memory():
    p = std_params(512, 512, T=20, K=16)
    z = np.zeros(4, np.float32)
    assert E.two_stage(p, z, z, np.array([0, 4], np.int64), 1, 1)["rc"] == -2


def test_restricted_theta_window():
    """theta window [pi/4, 3pi/4) -- the slopes within +-1 of the generator's tracks -- at the same angular
    resolution with half the rows (and half the votes); fast and general kernel against the oracle, records incl. the fp32 theta."""
    import math
    from dataclasses import replace
    wl = synth.workload(3)
    b = synth.generate(wl, 0, 3)
    p = replace(params_of(wl), n_theta=256, theta_min=math.pi / 4, theta_max=3 * math.pi / 4)
    o = oracle_run(p, b.u, b.v, b.offsets)
    for flags in (0, E.FLAG_GENERAL_ONLY):
        g = E.run(p, b.u, b.v, b.offsets, E.HOUGH_U16, flags=flags)
        assert_same(g, o, p)
        for e in range(3):
            k = min(int(o["n_found"][e]), p.max_candidates)
            assert g["cands"][e, :k].tobytes() == o["cands"][e, :k].tobytes()
    assert (o["cands"]["theta"][0, :8] >= math.pi / 4 - 1e-6).all() and (o["cands"]["theta"][0, :8] < 3 * math.pi / 4).all()


def test_dense_workload_is_handed_over_after_a_run_of_overflows():
    """2000 hits on a 128 x 128 grid switch (nearly) every bin on: each event overflows the fast kernel's lists.  After eight
    overflows in a row a CTA hands the next 64 events over without voting on them; results are the general kernel's either way."""
    wl = synth.workload(4, 2, 0)
    b = synth.generate(wl, 0, 30)
    p = params_of(wl)
    g = E.run(p, b.u, b.v, b.offsets, want_acc=False)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    assert_same(g, o, p)
    assert g["info"]["fast_groups"] > 0 and g["deferred"] == 30


def tiny_events(n_events, seed):
    """Many tiny events on a 64 x 64 grid: one short track (12 collinear hits) plus a few noise hits each."""
    rng = np.random.default_rng(seed)
    n = 16
    m, c = rng.uniform(-1, 1, n_events), rng.uniform(-100, 100, n_events)
    uu = np.tile(np.linspace(-90, 90, 12), (n_events, 1))
    vv = m[:, None] * uu + c[:, None]
    u = np.concatenate([uu, rng.uniform(-94, 94, (n_events, n - 12))], axis=1).astype(np.float32).ravel()
    v = np.concatenate([vv, rng.uniform(-194, 194, (n_events, n - 12))], axis=1).astype(np.float32).ravel()
    return u, v, np.arange(0, n * n_events + 1, n, dtype=np.int64)


def test_general_kernel_epoch_tags_wrap():
    """The general kernel tags its union-find words with a 10-bit per-CTA epoch instead of clearing its global scratch per event;
    after 1023 events of one CTA the tags would repeat, so the slab is cleared and the epoch restarts.  The model's first CTA
    takes every event: 1100 events cross that point."""
    p = std_params(64, 64, T=8, K=8)
    u, v, offsets = tiny_events(1100, seed=61)
    g = E.run(p, u, v, offsets, flags=E.FLAG_GENERAL_ONLY, want_acc=False)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert_same(g, o, p)
    assert (o["n_found"] >= 1).mean() > 0.9


# ----------------------------------------------------------------------------- theta wrap (reading B9)
def seam_events(n_events, seed, coord=94.0):
    """Events whose tracks are vertical or nearly so (theta within a few bins of 0 / pi: their ridges cross the seam) plus
    ordinary tracks and noise."""
    rng = np.random.default_rng(seed)
    us, vs, offs = [], [], [0]
    for e in range(n_events):
        uu, vv = [], []
        for k in range(int(rng.integers(1, 4))):                             # near-vertical: u = c + small slope * v
            c, tilt = rng.uniform(-0.9 * coord, 0.9 * coord), rng.uniform(-0.06, 0.06) if k else rng.uniform(-0.01, 0.01)
            v = rng.uniform(-190, 190, int(rng.integers(20, 48)) if k else 48)
            uu.append(np.clip(c + tilt * v + rng.normal(0, 0.1, len(v)), -coord, coord)); vv.append(v)
        for _ in range(int(rng.integers(0, 3))):                             # ordinary tracks
            a, b = synth.ideal_track(rng.uniform(-1, 1), rng.uniform(-100, 100))
            uu.append(a); vv.append(b)
        n_noise = int(rng.integers(0, 60))
        uu.append(rng.uniform(-coord, coord, n_noise)); vv.append(rng.uniform(-190, 190, n_noise))
        uu, vv = np.concatenate(uu).astype(np.float32), np.concatenate(vv).astype(np.float32)
        pm = rng.permutation(len(uu))
        us.append(uu[pm]); vs.append(vv[pm]); offs.append(offs[-1] + len(uu))
    return np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)


@pytest.mark.parametrize("grid,dt,K,T", [((256, 256), E.HOUGH_U16, 128, 10), ((1024, 256), E.HOUGH_U16, 64, 10),
                                        ((180, 1000), E.HOUGH_I32, 16, 4), ((45, 64), E.HOUGH_I32, 3, 10), ((3, 33), E.HOUGH_U16, 8, 10)],
                         ids=["256x256_u16", "1024x256_several_strips", "180x1000_i32", "45x64_K3", "three_rows"])
def test_theta_wrap_variant(grid, dt, K, T):
    """HOUGH_FLAG_THETA_WRAP: peaks and clusters that see across the theta seam, against the oracle with theta_wrap, and the
    same plan without the flag against the oracle without (the flag must change nothing else)."""
    u, v, offsets = seam_events(6, seed=grid[0])
    u = np.concatenate([u, np.zeros(0, np.float32)]); offsets = np.append(offsets, offsets[-1])    # an empty event at the end
    crossed = 0
    for wrap in (True, False):
        p = std_params(grid[0], grid[1], T=T, K=K, theta_wrap=wrap)
        g = E.run(p, u, v, offsets, dt, want_acc=False)
        o = oracle_run(p, u, v, offsets, want_acc=False)
        assert_same(g, o, p)
        assert g["info"]["fast_groups"] == 0 or not wrap                    # wrap plans use the general kernel
        if wrap:
            o_plain = oracle_run(std_params(grid[0], grid[1], T=10, K=K), u, v, offsets, want_acc=False)
            crossed = sum(int(o["n_found"][e] != o_plain["n_found"][e] or o["cands"][e].tobytes() != o_plain["cands"][e].tobytes())
                          for e in range(len(offsets) - 1))
    assert crossed >= (1 if grid[0] >= 45 else 0)                            # the seam really matters on these events


def test_theta_wrap_is_rejected_where_the_seam_does_not_close():
    ok = std_params(64, 64)
    for bad in (dict(rho_min=-256.0, rho_max=300.0), dict(n_theta=2), dict(theta_min=0.0, theta_max=1.5)):
        p = std_params(**{**dict(n_theta=64, n_rho=64), **bad})
        d = E.Desc(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, 6, -1, 5, 2.0, 8, E.HOUGH_I32, 1, 10, 10, E.FLAG_THETA_WRAP, 0,
                   *E.theta_window(p))
        h = E.ctypes.c_void_p()
        assert E.lib().hough_plan_create(E.ctypes.byref(d), E.ctypes.byref(h)) == -1
    d = E.Desc(ok.n_theta, ok.n_rho, ok.rho_min, ok.rho_max, ok.coord_max, 6, -1, 5, 2.0, 8, E.HOUGH_I32, 1, 10, 10, E.FLAG_THETA_WRAP, 0, 0.0, 0.0)
    h = E.ctypes.c_void_p()
    assert E.lib().hough_plan_create(E.ctypes.byref(d), E.ctypes.byref(h)) == 0
    z = E.DevBuf(np.zeros(4, np.float32)); off = E.DevBuf(np.array([0, 4], np.int64))
    cands = E.DevBuf(np.zeros((1, 8), E.CAND_DTYPE)); nf = E.DevBuf(np.zeros(1, np.int32)); lab = E.DevBuf(np.zeros(4, np.int32))
    L = E.lib()
    L.hough_find_tracks_peeloff.argtypes = [E.ctypes.c_void_p] * 4 + [E.ctypes.c_int32] + [E.ctypes.c_void_p] * 4
    L.hough_find_two_stage.argtypes = [E.ctypes.c_void_p] * 4 + [E.ctypes.c_int32] * 3 + [E.ctypes.c_void_p] * 3
    assert L.hough_find_tracks_peeloff(h, z.ptr, z.ptr, off.ptr, 1, cands.ptr, nf.ptr, lab.ptr, None) == -1
    assert L.hough_find_two_stage(h, z.ptr, z.ptr, off.ptr, 1, 4, 4, cands.ptr, nf.ptr, None) == -1
    L.hough_plan_destroy(h)


@pytest.mark.parametrize("seed,preempt,workers", [(11, 0, 1), (12, 64, 1), (13, 8, 4)])
def test_theta_wrap_does_not_depend_on_the_schedule(seed, preempt, workers):
    u, v, offsets = seam_events(8, seed=5)
    p = std_params(256, 128, T=10, K=32, theta_wrap=True)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    E.configure(seed=seed, preempt_per_1024=preempt, workers=workers)
    assert_same(E.run(p, u, v, offsets, E.HOUGH_U16, want_acc=False), o, p)


# ----------------------------------------------------------------------------- caller data that names nothing of the plan
def test_assign_ignores_records_that_name_no_bin_of_the_plan():
    """hough_assign_hits on records the caller made up: slots whose (theta_bin, rho_bin) lie outside the grid must not index the
    tables (on the GPU: an out-of-range read); they attract no hit, and the good slots label exactly as the oracle says."""
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 6)
    p = params_of(wl)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    cands = o["cands"].copy()
    n_found = o["n_found"].copy()
    bad_slots = {}
    for e in range(6):
        nk = min(int(n_found[e]), p.max_candidates)
        if nk >= 2:
            s = nk - 1                                                       # the last kept record becomes garbage
            cands[e, s]["theta_bin"], cands[e, s]["rho_bin"] = [(-1, 5), (p.n_theta, 0), (3, -7), (2 ** 30, 2 ** 30), (0, p.n_rho), (-2 ** 31, 1)][e]
            bad_slots[e] = s
    assert bad_slots
    labels, rc, rc_null = E.assign(p, b.u, b.v, b.offsets, cands, n_found)
    assert rc == 0 and rc_null == -1                                         # a null labels pointer is refused, not written through
    for e in range(6):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        nk = min(int(n_found[e]), p.max_candidates)
        good = [c for s, c in enumerate(o["cands"][e, :nk]) if s != bad_slots.get(e)]
        want = C.assign_event(b.u[a:z], b.v[a:z], np.array(good, C.CAND_DTYPE), p)   # slots keep their numbers: the bad one is the last
        np.testing.assert_array_equal(labels[a:z], want)
        assert bad_slots.get(e, -5) not in set(labels[a:z].tolist())


def test_refit_ignores_labels_beyond_the_kept_records():
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 5)
    p = params_of(wl)
    o = C.run_batch(b.u, b.v, b.offsets, p)
    labels = o["labels"].copy()
    labels[::7] = np.array([p.max_candidates, 2 ** 30, 99, 4096], np.int32)[np.arange(len(labels[::7])) % 4]   # made-up slots
    fits, rc = E.refit(p, b.u, b.v, b.offsets, o["n_found"], labels, GEOM)
    assert rc == 0
    for e in range(5):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        nk = min(int(o["n_found"][e]), p.max_candidates)
        lab = labels[a:z].copy()
        lab[lab >= nk] = -1                                                  # what "ignored" means
        fits_equal(fits[e], T.refit_event(b.u[a:z], b.v[a:z], lab, nk, p, GEOM))


@pytest.mark.parametrize("flags", [0, E.FLAG_GENERAL_ONLY], ids=["fast", "general_only"])
def test_an_event_that_ends_beyond_the_plans_hit_capacity_is_flagged_not_read(flags):
    """offsets[e + 1] > max_hits: the hits of that event would be read past the caller's buffers (the model ends them at an
    inaccessible page).  The event is flagged BAD_OFFSETS and skipped by every kernel; its neighbours are computed."""
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 3)
    p = params_of(wl)
    n = len(b.u)
    offsets = b.offsets.copy()
    offsets[3] = n + 50                                                      # the last event claims 50 hits that do not exist
    g = E.run(p, b.u, b.v, offsets, flags=flags, want_vote=False)           # E.run sizes the plan by len(u): max_hits = n
    assert g["emu_violations"] == 0 and g["bounds_violations"] == 0
    assert g["status"] == 2
    o = C.run_batch(b.u, b.v, b.offsets, p)
    np.testing.assert_array_equal(g["n_found"][:2], o["n_found"][:2])
    assert g["n_found"][2] == 0
    a = int(b.offsets[2])
    np.testing.assert_array_equal(g["labels"][:a], o["labels"][:a])
    assert (g["labels"][a:] == -99).all()                                    # untouched
    fits, rc = E.refit(p, b.u, b.v, offsets, g["n_found"], np.where(g["labels"] == -99, -1, g["labels"]), GEOM)
    assert rc == 0 and (fits[2]["n_hits"] == 0).all()
    pe = E.peeloff(std_params(64, 64, T=8, K=4), b.u, b.v, offsets, max_hpe=int(np.diff(offsets).max()))
    assert pe["status"] == 2 and pe["n_found"][2] == 0
    ts = E.two_stage(std_params(64, 64, T=8, K=4), b.u, b.v, offsets, 4, 4)
    assert ts["rc"] == 0 and ts["n_found"][2] == 0


def test_frontend_skips_fills_whose_range_is_not_inside_the_hits():
    """Fill offsets are caller data: a fill that starts below 0, ends before it starts or ends beyond n_hits is skipped and flagged
    (BAD_OFFSETS); it is never used to index the per-hit scratch (found by tests/emu/fuzz_hostile.py: an endless loop otherwise)."""
    fe = T.FrontEnd(windows_per_fill=6)
    x, y, z, t, fo = synthetic_fills(4, seed=44)
    n = len(x)
    for bad in ([0, int(fo[1]), n + 100, int(fo[3]), n], [0, -5, int(fo[2]), int(fo[3]), n], [0, int(fo[2]), int(fo[1]), int(fo[3]), 2 ** 40]):
        g = E.frontend_slice(fe, x, y, z, t, np.array(bad, np.int64))
        assert g["status"] & 2
    g = E.frontend_slice(fe, x, y, z, t, fo)                                 # and the honest offsets are not flagged
    assert g["status"] == 0
