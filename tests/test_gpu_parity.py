"""GPU parity: the CUDA path (through the C ABI of include/hough.h) against the CPU oracle, element by element,
on the same seeded inputs.  Everything integer is compared bit-exactly; the two fp32 line parameters within
1e-5 relative (BASELINE.json north_star).  Run on the B200 box: python -m pytest tests -m gpu."""
import numpy as np
import pytest
import torch

from oracle import hough_c as C
from oracle import hough_def as D
from paper_2511_02742_b200 import hough as H
from paper_2511_02742_b200 import synth
from test_oracle_pins import edge_cases
from util import mixed_batch, paper_grid_batch, params_of, std_params

pytestmark = pytest.mark.gpu

INT_FIELDS = ("theta_bin", "rho_bin", "votes", "cluster_root", "cluster_nbins", "reserved")


def make_plan(p: D.Params, n_events, n_hits, max_hpe, count_dtype=H.HOUGH_I32, flags=0):
    if p.theta_wrap:
        flags |= H.HOUGH_FLAG_THETA_WRAP
    return H.hough_plan_create(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window,
                               p.max_candidates, max(1, n_events), max(0, n_hits), max_hpe, count_dtype,
                               p.hit_frac_bits, p.acc_frac_bits, 0, flags,
                               *((0.0, 0.0) if (p.theta_min == 0.0 and p.theta_max == np.pi) else (p.theta_min, p.theta_max)))


def gpu_run(p: D.Params, u, v, offsets, count_dtype=H.HOUGH_I32, want_acc=True, max_hpe=None, flags=0, want_vote=True):
    """Whole CUDA path on one batch; returns numpy results shaped like oracle.hough_c.run_batch, plus which kernel did the
    work: info["fast_groups"] (0 = the plan has no fast kernel) and "deferred" (events the fast kernel handed over)."""
    E = len(offsets) - 1
    hpe = int(np.diff(offsets).max()) if E > 0 and len(u) else 0
    plan = make_plan(p, E, len(u), max(hpe, 1) if max_hpe is None else max_hpe, count_dtype, flags)
    du = torch.from_numpy(np.ascontiguousarray(u, np.float32)).cuda()
    dv = torch.from_numpy(np.ascontiguousarray(v, np.float32)).cuda()
    do = torch.from_numpy(np.ascontiguousarray(offsets, np.int64)).cuda()
    out = {}
    acc = dig = None
    if want_vote:
        acc, dig = H.hough_vote(plan, du, dv, do, want_acc=want_acc, want_digest=True)
    cands, n_found = H.hough_find_clusters(plan, du, dv, do)
    labels = H.hough_assign_hits(plan, du, dv, do, cands, n_found)
    torch.cuda.synchronize()
    dbg = H.hough_plan_debug_counters(plan)
    out["deferred"], out["bounds_violations"], out["bounds_site"] = int(dbg[15]), int(dbg[14]), int(dbg[13])
    out["status"] = H.hough_plan_status(plan)
    if acc is not None:
        a = acc.cpu().numpy()
        out["acc"] = a.view(np.uint16).astype(np.int32) if a.dtype == np.int16 else a
    if dig is not None:
        out["digest"] = dig.cpu().numpy().view(np.uint64)
    out["cands"] = H.candidates_to_numpy(cands)
    out["n_found"] = n_found.cpu().numpy()
    out["labels"] = labels.cpu().numpy()
    out["info"] = H.hough_plan_query(plan)[0]
    H.hough_plan_destroy(plan)
    return out


def assert_same(g, o, p: D.Params, check_acc=True, status=0):
    assert g["bounds_violations"] == 0, f"index check failed inside a kernel, first at site {g['bounds_site']}"
    assert g["status"] == status
    if check_acc and "acc" in g:
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


def assert_path(g, fast: bool, deferred=None):
    """Which kernel produced the result: the plan has (no) fast kernel; `deferred` = 0, an exact count, or ">0"."""
    assert (g["info"]["fast_groups"] > 0) == fast, g["info"]
    if deferred == ">0":
        assert g["deferred"] > 0
    elif deferred is not None:
        assert g["deferred"] == deferred, g["deferred"]


# ----------------------------------------------------------------------------- tables first (libm check)
@pytest.mark.parametrize("grid", [(180, 256), (256, 256), (256, 512), (512, 512), (128, 128), (1024, 1024), (180, 1000)])
def test_tables_and_constants_equal_oracle(grid):
    p = std_params(*grid) if grid != (180, 1000) else D.Params(180, 1000, -500.0, 500.0, 360.0, 6, 1.0, 16)
    plan = make_plan(p, 1, 100, 100)
    info, cq, sq = H.hough_plan_query(plan)
    Hh, F, Oq, Wq, Cq, Sq = C.constants(p)
    assert (info["hit_frac_bits"], info["acc_frac_bits"], info["rho_offset_q"], info["assign_window_q"]) == (Hh, F, Oq, Wq)
    np.testing.assert_array_equal(cq.astype(np.int64), Cq)
    np.testing.assert_array_equal(sq.astype(np.int64), Sq)
    H.hough_plan_destroy(plan)


# ----------------------------------------------------------------------------- BASELINE configs at oracle-sized samples
@pytest.mark.gate
@pytest.mark.parametrize("cfg,n_events", [(0, 1), (1, 8), (2, 4), (3, 3)])
def test_gate_configs_small(cfg, n_events):
    """The first thing an untested build runs: at most 8 events per config."""
    wl = synth.workload(cfg)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    dt = H.HOUGH_U16 if wl.count_dtype == "u16" else H.HOUGH_I32
    for flags, fast, deferred in ((0, True, 0), (H.HOUGH_FLAG_SMALL_LISTS, True, None), (H.HOUGH_FLAG_GENERAL_ONLY, False, 0)):
        g = gpu_run(p, b.u, b.v, b.offsets, dt, flags=flags)
        o = oracle_run(p, b.u, b.v, b.offsets)
        assert_same(g, o, p)
        assert_path(g, fast, deferred)


@pytest.mark.parametrize("cfg,n_events", [(0, 1), (1, 96), (2, 40), (3, 12)])
def test_configs_bit_exact(cfg, n_events):
    wl = synth.workload(cfg)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    dt = H.HOUGH_U16 if wl.count_dtype == "u16" else H.HOUGH_I32
    g = gpu_run(p, b.u, b.v, b.offsets, dt)
    o = oracle_run(p, b.u, b.v, b.offsets)
    assert_same(g, o, p)
    assert_path(g, fast=True, deferred=0)              # S1-S4 of these events ran in the fast kernel
    assert g["acc"].sum() == b.n_hits * wl.n_theta     # P4: every generator hit votes once per theta row


@pytest.mark.parametrize("cfg,n_events", [(1, 2400), (3, 640)])
def test_many_events_per_cta_fast_kernel(cfg, n_events):
    """More events than 4 x the persistent CTAs: every CTA processes several events back to back (per-event reset of halos,
    lists and histogram, tile reuse, work counter).  Digests prove the accumulators, records and labels the rest."""
    wl = synth.workload(cfg)
    wl = wl.with_events(max(wl.n_events, n_events))      # cfg1 lists 1000 events: further chunks of the same stream
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    dt = H.HOUGH_U16 if wl.count_dtype == "u16" else H.HOUGH_I32
    g = gpu_run(p, b.u, b.v, b.offsets, dt, want_acc=False)
    assert n_events >= 4 * g["info"]["fast_ctas"]
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    assert_same(g, o, p)
    assert_path(g, fast=True, deferred=0)


def test_mixed_batch_with_deferred_events_interleaved():
    wl, u, v, offsets, kinds = mixed_batch(1, 1500, seed=21)
    p = params_of(wl)
    n_big = kinds.count("count>1023")
    assert n_big >= 10 and kinds.count("empty") >= 20
    g = gpu_run(p, u, v, offsets, want_acc=False, max_hpe=2048)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert_same(g, o, p)
    assert_path(g, fast=True, deferred=n_big)          # exactly the events with a count above 1023 were handed over
    big = kinds.index("count>1023")
    assert o["cands"][big, 0]["votes"] == 1100


def test_events_longer_than_the_fast_staging_buffer_are_deferred():
    wl, u, v, offsets, kinds = mixed_batch(2, 300, seed=22, long_hits=9000)
    p = params_of(wl)
    n_long = kinds.count("long")
    assert n_long >= 2
    g = gpu_run(p, u, v, offsets, want_acc=False, max_hpe=9000)
    assert g["info"]["fast_hits_cap"] < 9000
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert_same(g, o, p)
    assert_path(g, fast=True, deferred=n_long + kinds.count("count>1023"))


@pytest.mark.parametrize("cfg,n_events", [(1, 400), (3, 160)])
def test_small_lists_force_the_hand_over(cfg, n_events):
    """HOUGH_FLAG_SMALL_LISTS: ordinary events overflow the fast kernel's lists mid-way (strip list, on list, peak list) and
    are recomputed by the general kernel; results stay identical."""
    wl = synth.workload(cfg)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    dt = H.HOUGH_U16 if wl.count_dtype == "u16" else H.HOUGH_I32
    g = gpu_run(p, b.u, b.v, b.offsets, dt, want_acc=False, flags=H.HOUGH_FLAG_SMALL_LISTS)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    assert_same(g, o, p)
    assert_path(g, fast=True, deferred=">0")


@pytest.mark.parametrize("cfg,n_events", [(1, 700), (3, 40)])
def test_general_kernel_alone(cfg, n_events):
    wl = synth.workload(cfg)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    dt = H.HOUGH_U16 if wl.count_dtype == "u16" else H.HOUGH_I32
    g = gpu_run(p, b.u, b.v, b.offsets, dt, want_acc=False, flags=H.HOUGH_FLAG_GENERAL_ONLY)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    assert_same(g, o, p)
    assert_path(g, fast=False, deferred=0)


def test_paper_grid_180x1000_multi_event():
    """The paper's own CPU grid (180 theta bins over 0-180 deg, 1000 rho bins over -500...500), 40 planes
    (L72 "40 vanes"), a batch of events."""
    p, u, v, offsets = paper_grid_batch(200)
    g = gpu_run(p, u, v, offsets, want_acc=False)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert_same(g, o, p)
    assert (o["n_found"] >= 1).mean() > 0.8            # (a track steeper than the rho range allows can go unseen)


@pytest.mark.parametrize("hits_idx", [0, 1, 2, 3])
@pytest.mark.parametrize("grid_idx", [0, 1, 2, 3])
def test_config4_cells_bit_exact(hits_idx, grid_idx):
    """All 16 cells of the roofline sweep (hits/event x grid), enough events that CTAs of the fast kernel take several."""
    wl = synth.workload(4, hits_idx, grid_idx)
    n_events = {0: 320, 1: 160, 2: 24, 3: 6}[hits_idx] if grid_idx < 3 else {0: 40, 1: 24, 2: 8, 3: 3}[hits_idx]
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    g = gpu_run(p, b.u, b.v, b.offsets, want_acc=(n_events <= 24 and grid_idx < 3))
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=(n_events <= 24 and grid_idx < 3))
    assert_same(g, o, p)


# ----------------------------------------------------------------------------- adversarial edge set
@pytest.mark.gate
@pytest.mark.parametrize("case", edge_cases(), ids=lambda c: c[0])
def test_edge_set(case):
    name, p, u, v = case
    offsets = np.array([0, len(u)], np.int64)
    g = gpu_run(p, u, v, offsets, max_hpe=max(len(u), 1))
    o = oracle_run(p, u, v, offsets)
    assert_same(g, o, p)


@pytest.mark.gate
def test_edge_set_as_one_ragged_batch():
    """Same grid cases concatenated into one batch with empty events in between (ragged offsets, unaligned starts)."""
    cases = [c for c in edge_cases() if c[1] == edge_cases()[0][1]]
    p = cases[0][1]
    us, vs, offs = [], [], [0]
    for _, _, u, v in cases:
        us.append(u); vs.append(v); offs.append(offs[-1] + len(u)); offs.append(offs[-1])    # + an empty event
    u, v, offsets = np.concatenate(us), np.concatenate(vs), np.array(offs, np.int64)
    g = gpu_run(p, u, v, offsets)
    o = oracle_run(p, u, v, offsets)
    assert_same(g, o, p)


def test_u16_boundary_65535_identical_hits():
    p = std_params(8, 16, T=65535, K=4)
    u = np.full(65535, 3.0, np.float32)
    v = np.full(65535, 5.0, np.float32)
    offsets = np.array([0, 65535], np.int64)
    g = gpu_run(p, u, v, offsets, H.HOUGH_U16)
    o = oracle_run(p, u, v, offsets)
    assert_same(g, o, p)
    assert g["acc"].max() == 65535


def test_more_than_65535_hits_uses_wide_counters():
    p = std_params(32, 32, T=60000, K=4)
    n = 70000
    rng = np.random.default_rng(5)
    u = np.where(rng.random(n) < 0.9, 3.0, rng.uniform(-200, 200, n)).astype(np.float32)
    v = np.where(rng.random(n) < 0.9, 5.0, rng.uniform(-200, 200, n)).astype(np.float32)
    offsets = np.array([0, n], np.int64)
    g = gpu_run(p, u, v, offsets)
    assert g["info"]["counter_bytes"] == 4
    o = oracle_run(p, u, v, offsets)
    assert_same(g, o, p)


def test_many_hits_per_event_is_staged_in_chunks():
    wl = synth.workload(4, 3, 1)                      # 8000 hits / event > the 4096-hit staging buffer
    b = synth.generate(wl, 0, 3)
    p = params_of(wl, max_candidates=16)
    g = gpu_run(p, b.u, b.v, b.offsets)
    o = oracle_run(p, b.u, b.v, b.offsets)
    assert_same(g, o, p)


def test_unsafe_hits_near_the_rho_range_edge():
    """Hits whose sinusoid leaves [rho_min, rho_max): the range-checked vote path; out-of-range votes are dropped."""
    rng = np.random.default_rng(11)
    p = std_params(256, 256, T=4, K=64)
    u = rng.uniform(-256, 256, 600).astype(np.float32)
    v = rng.uniform(-256, 256, 600).astype(np.float32)
    offsets = np.array([0, 100, 100, 350, 600], np.int64)
    g = gpu_run(p, u, v, offsets)
    o = oracle_run(p, u, v, offsets)
    assert_same(g, o, p)
    assert g["acc"].sum() < 600 * 256                 # some votes really were out of range


def test_strip_seams_dense_mask():
    """A dense on-mask (low threshold, many hits): clusters and maxima that straddle every strip seam."""
    rng = np.random.default_rng(12)
    p = std_params(512, 512, T=3, K=128)
    u = rng.uniform(-94, 94, 1500).astype(np.float32)
    v = rng.uniform(-194, 194, 1500).astype(np.float32)
    offsets = np.array([0, 700, 1500], np.int64)
    g = gpu_run(p, u, v, offsets, want_acc=True)
    o = oracle_run(p, u, v, offsets)
    assert g["info"]["n_strips"] >= 2
    assert_same(g, o, p)


def test_large_K_and_overflowing_peak_list():
    rng = np.random.default_rng(13)
    p = std_params(512, 512, T=1, K=4096)
    u = rng.uniform(-94, 94, 300).astype(np.float32)
    v = rng.uniform(-194, 194, 300).astype(np.float32)
    offsets = np.array([0, 300], np.int64)
    g = gpu_run(p, u, v, offsets, want_acc=False)
    o = oracle_run(p, u, v, offsets)
    assert o["n_found"][0] > 4096
    assert_same(g, o, p)


def test_permutation_invariance_on_gpu():
    wl = synth.workload(2)
    b = synth.generate(wl, 0, 4)
    p = params_of(wl)
    g1 = gpu_run(p, b.u, b.v, b.offsets)
    rng = np.random.default_rng(3)
    u2, v2 = b.u.copy(), b.v.copy()
    perms = []
    for e in range(b.n_events):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        pm = rng.permutation(z - a)
        perms.append(pm)
        u2[a:z], v2[a:z] = b.u[a:z][pm], b.v[a:z][pm]
    g2 = gpu_run(p, u2, v2, b.offsets)
    np.testing.assert_array_equal(g1["acc"], g2["acc"])
    np.testing.assert_array_equal(g1["n_found"], g2["n_found"])
    assert g1["cands"].tobytes() == g2["cands"].tobytes()
    for e, pm in enumerate(perms):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        np.testing.assert_array_equal(g1["labels"][a:z][pm], g2["labels"][a:z])


def test_status_word_flags_long_events_and_bad_offsets():
    p = std_params(64, 64, T=3, K=8)
    rng = np.random.default_rng(2)
    u = rng.uniform(-100, 100, 300).astype(np.float32)
    v = rng.uniform(-100, 100, 300).astype(np.float32)
    offsets = np.array([0, 50, 250, 300], np.int64)             # middle event has 200 hits > capacity 100
    g = gpu_run(p, u, v, offsets, max_hpe=100)
    assert g["status"] & H.HOUGH_STATUS_EVENT_TOO_LONG
    assert g["n_found"][1] == 0 and (g["labels"][50:250] == -1).all()
    o = C.run_batch(u[:50], v[:50], np.array([0, 50], np.int64), p)
    np.testing.assert_array_equal(g["labels"][:50], o["labels"])


def test_an_event_that_ends_beyond_the_plans_hit_capacity_is_flagged_not_read():
    """offsets[e + 1] > max_hits: BAD_OFFSETS, the event is skipped by every kernel (its hits would lie past the buffers)."""
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 3)
    p = params_of(wl)
    n = len(b.u)
    offsets = b.offsets.copy()
    offsets[3] = n + 50
    o = C.run_batch(b.u, b.v, b.offsets, p)
    a = int(b.offsets[2])
    for flags in (0, H.HOUGH_FLAG_GENERAL_ONLY):
        plan = make_plan(p, 3, n, int(np.diff(offsets).max()), H.HOUGH_I32, flags)        # max_hits = n
        du, dv = torch.from_numpy(b.u).cuda(), torch.from_numpy(b.v).cuda()
        do = torch.from_numpy(offsets).cuda()
        cands, n_found = H.hough_find_clusters(plan, du, dv, do)
        labels = torch.full((n,), -99, dtype=torch.int32, device="cuda")
        H.hough_assign_hits(plan, du, dv, do, cands, n_found, labels=labels)
        torch.cuda.synchronize()
        assert H.hough_plan_status(plan) == H.HOUGH_STATUS_BAD_OFFSETS
        nf, lab = n_found.cpu().numpy(), labels.cpu().numpy()
        np.testing.assert_array_equal(nf[:2], o["n_found"][:2])
        assert nf[2] == 0 and (lab[a:] == -99).all()
        np.testing.assert_array_equal(lab[:a], o["labels"][:a])
        H.hough_plan_destroy(plan)


def test_assign_ignores_records_that_name_no_bin_of_the_plan():
    """Records are caller data: slots whose bin lies just outside the grid must not index the tables and attract no hit."""
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 6)
    p = params_of(wl)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    cands = o["cands"].copy()
    bad_slots = {}
    for e in range(6):
        nk = min(int(o["n_found"][e]), p.max_candidates)
        if nk >= 2:
            cands[e, nk - 1]["theta_bin"], cands[e, nk - 1]["rho_bin"] = [(-1, 5), (p.n_theta, 0), (3, -7), (1, p.n_rho), (0, p.n_rho + 3), (-2, 1)][e]
            bad_slots[e] = nk - 1
    assert bad_slots
    plan = make_plan(p, 6, len(b.u), int(np.diff(b.offsets).max()))
    du, dv, do = torch.from_numpy(b.u).cuda(), torch.from_numpy(b.v).cuda(), torch.from_numpy(b.offsets).cuda()
    dc = torch.from_numpy(np.ascontiguousarray(cands).view(np.int32).reshape(6, p.max_candidates, 8)).cuda()
    dn = torch.from_numpy(o["n_found"]).cuda()
    labels = H.hough_assign_hits(plan, du, dv, do, dc, dn).cpu().numpy()
    H.hough_plan_destroy(plan)
    for e in range(6):
        a, z = int(b.offsets[e]), int(b.offsets[e + 1])
        nk = min(int(o["n_found"][e]), p.max_candidates)
        good = np.array([c for s, c in enumerate(o["cands"][e, :nk]) if s != bad_slots.get(e)], C.CAND_DTYPE)
        np.testing.assert_array_equal(labels[a:z], C.assign_event(b.u[a:z], b.v[a:z], good, p))


@pytest.mark.parametrize("n_chunks,n_events", [(0, 32), (1, 32), (3, 500), (7, 500), (32, 40)])
def test_run_host_chunked_equals_oracle(n_chunks, n_events):
    """hough_run_host / hough_run_host_chunked: the three-stream chunk pipeline (upload, compute, download), called twice on
    one plan; chunk boundaries fall inside the batch, with empty events around them."""
    wl = synth.workload(1)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    offsets = np.concatenate([b.offsets[:n_events // 2], np.repeat(b.offsets[n_events // 2], 3), b.offsets[n_events // 2:]])  # + 3 empty events
    E = len(offsets) - 1
    plan = make_plan(p, E, b.n_hits, int(np.diff(offsets).max()))
    o = C.run_batch(b.u, b.v, offsets, p)
    for rep in range(2):
        cands = np.zeros((E, p.max_candidates, 8), np.int32)
        n_found = np.full(E, -7, np.int32)
        labels = np.full(b.n_hits, -7, np.int32)
        before = H.hough_plan_launch_count(plan)
        H.hough_run_host(plan, b.u, b.v, offsets, cands, n_found, labels, n_chunks=n_chunks)
        chunks_run = (H.hough_plan_launch_count(plan) - before) // 3    # fast + general-on-deferred + assign per chunk
        want = 1 if n_chunks == 0 else min(n_chunks, E)
        assert chunks_run == want if want <= 7 else 1 <= chunks_run <= want     # (a chunk without events launches nothing)
        np.testing.assert_array_equal(n_found, o["n_found"])
        np.testing.assert_array_equal(labels, o["labels"])
        gc = cands.view(H.CANDIDATE_DTYPE).reshape(E, p.max_candidates)
        for e in range(E):
            k = min(int(n_found[e]), p.max_candidates)
            for f in INT_FIELDS:
                np.testing.assert_array_equal(gc[e, :k][f], o["cands"][e, :k][f])
    assert H.hough_plan_status(plan) == 0
    H.hough_plan_destroy(plan)


def test_bad_arguments_are_rejected_not_crashed():
    with pytest.raises(H.HoughError) as ei:
        H.hough_plan_create(0, 256, -256, 256, 256, 24, 2.0, 128, 10, 1000, 500)
    assert ei.value.status == H.HOUGH_EINVAL
    with pytest.raises(H.HoughError) as ei:
        H.hough_plan_create(256, 256, -256, 256, 256, 24, 2.0, 128, 10, 1000, 500, acc_frac_bits=28)   # int32 proof fails
    assert ei.value.status == H.HOUGH_ERANGE
    with pytest.raises(H.HoughError) as ei:
        H.hough_plan_create(256, 256, -256, 256, 256, 24, 2.0, 128, 10, 1000, 70000, count_dtype=H.HOUGH_U16)
    assert ei.value.status == H.HOUGH_ERANGE
    plan = H.hough_plan_create(64, 64, -256, 256, 256, 3, 8.0, 8, 4, 1000, 500)
    u = torch.zeros(1001, device="cuda")[1:]                    # misaligned (4-byte offset) hit array
    off = torch.tensor([0, 10], dtype=torch.int64, device="cuda")
    with pytest.raises(H.HoughError) as ei:
        H.hough_find_clusters(plan, u, u, off)
    assert ei.value.status == H.HOUGH_EINVAL
    off_big = torch.zeros(6, dtype=torch.int64, device="cuda")  # 5 events > max_events 4
    with pytest.raises(H.HoughError) as ei:
        H.hough_find_clusters(plan, torch.zeros(8, device="cuda"), torch.zeros(8, device="cuda"), off_big)
    assert ei.value.status == H.HOUGH_ERANGE
    H.hough_plan_destroy(plan)


def test_restricted_theta_window():
    """theta window [pi/4, 3pi/4) at the resolution of cfg3 with half the rows; records incl. the fp32 theta."""
    from dataclasses import replace
    wl = synth.workload(3)
    b = synth.generate(wl, 0, 200)
    p = replace(params_of(wl), n_theta=256, theta_min=np.pi / 4, theta_max=3 * np.pi / 4)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    for flags in (0, H.HOUGH_FLAG_GENERAL_ONLY):
        g = gpu_run(p, b.u, b.v, b.offsets, H.HOUGH_U16, want_acc=False, flags=flags)
        assert_same(g, o, p)
        for e in range(200):
            k = min(int(o["n_found"][e]), p.max_candidates)
            assert g["cands"][e, :k].tobytes() == o["cands"][e, :k].tobytes()


@pytest.mark.parametrize("grid,dt,K,T,n_events", [((256, 256), H.HOUGH_U16, 128, 10, 400), ((1024, 256), H.HOUGH_U16, 64, 10, 300),
                                                 ((180, 1000), H.HOUGH_I32, 16, 4, 300), ((45, 64), H.HOUGH_I32, 3, 10, 400),
                                                 ((3, 33), H.HOUGH_U16, 8, 10, 100)],
                         ids=["256x256_u16", "1024x256_several_strips", "180x1000_i32", "45x64_K3", "three_rows"])
def test_theta_wrap_variant(grid, dt, K, T, n_events):
    """SURVEY.md 8(f) item 4, reading B9 (HOUGH_FLAG_THETA_WRAP): peaks and clusters that see across the theta seam, on events
    whose near-vertical tracks put their ridges across it; every record and label against the oracle with theta_wrap."""
    from test_emulated_kernels import seam_events
    u, v, offsets = seam_events(n_events, seed=grid[0] + 1)
    p = std_params(grid[0], grid[1], T=T, K=K, theta_wrap=True)
    g = gpu_run(p, u, v, offsets, dt, want_acc=False)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    assert_same(g, o, p)
    assert g["info"]["fast_groups"] == 0                                     # wrap plans use the general kernel
    for e in range(n_events):
        k = min(int(o["n_found"][e]), p.max_candidates)
        assert g["cands"][e, :k].tobytes() == o["cands"][e, :k].tobytes()
    o_plain = oracle_run(std_params(grid[0], grid[1], T=T, K=K), u, v, offsets, want_acc=False)
    differ = sum(o["cands"][e].tobytes() != o_plain["cands"][e].tobytes() for e in range(n_events))
    assert differ >= (n_events // 10 if grid[0] >= 45 else 0)                # the seam matters on these events


def test_theta_wrap_on_the_high_pileup_grid():
    """The wrap variant on the events and the grid of config 3 (the benchmark workload)."""
    from dataclasses import replace
    wl = synth.workload(3)
    b = synth.generate(wl, 0, 60)
    p = replace(params_of(wl), theta_wrap=True)
    o = oracle_run(p, b.u, b.v, b.offsets, want_acc=False)
    g = gpu_run(p, b.u, b.v, b.offsets, H.HOUGH_U16, want_acc=False)
    assert_same(g, o, p)


def test_theta_wrap_is_rejected_where_the_seam_does_not_close():
    for bad in (dict(rho_min=-256.0, rho_max=300.0), dict(n_theta=2), dict(theta_min=0.0, theta_max=1.5)):
        p = std_params(**{**dict(n_theta=64, n_rho=64, theta_wrap=True), **bad})
        with pytest.raises(Exception):
            make_plan(p, 1, 16, 16)
    plan = make_plan(std_params(64, 64, theta_wrap=True), 1, 16, 16)
    z = torch.zeros(4, dtype=torch.float32, device="cuda")
    off = torch.tensor([0, 4], dtype=torch.int64, device="cuda")
    with pytest.raises(Exception):
        H.hough_find_tracks_peeloff(plan, z, z, off)
    with pytest.raises(Exception):
        H.hough_find_two_stage(plan, z, z, off, 4, 4)
    H.hough_plan_destroy(plan)


def test_general_kernel_epoch_tags_wrap():
    """More than 1023 events per persistent CTA through the general kernel: its 10-bit epoch tags wrap, the per-CTA union-find
    slab is cleared and the epoch restarts.  320,000 tiny events: more than 1023 per CTA on average even with 296 CTAs."""
    from test_emulated_kernels import tiny_events
    p = std_params(64, 64, T=8, K=8)
    n = 320000
    u, v, offsets = tiny_events(n, seed=62)
    g = gpu_run(p, u, v, offsets, want_vote=False, flags=H.HOUGH_FLAG_GENERAL_ONLY)
    assert g["info"]["n_ctas"] * 1023 < n and g["bounds_violations"] == 0 and g["status"] == 0
    assert_path(g, fast=False, deferred=0)
    o = oracle_run(p, u, v, offsets, want_acc=False)
    np.testing.assert_array_equal(g["n_found"], o["n_found"])
    np.testing.assert_array_equal(g["labels"], o["labels"])
    kept = np.arange(p.max_candidates)[None, :] < np.minimum(o["n_found"], p.max_candidates)[:, None]
    for f in INT_FIELDS + ("theta", "rho"):
        np.testing.assert_array_equal(g["cands"][f][kept], o["cands"][f][kept], err_msg=f)


# ----------------------------------------------------------------------------- BASELINE sizes, bench.py's launch configuration
def _gen_chunk(job):
    from paper_2511_02742_b200 import synth as S
    b = S.generate_chunk(job[0], job[1])
    return b.u, b.v, b.offsets


def generate_all(wl, n_events):
    """The first n_events events of a workload, chunks generated in worker processes (spawned: CUDA is alive in this one)."""
    import multiprocessing as mp
    import os
    n_chunks = (n_events + synth.CHUNK_EVENTS - 1) // synth.CHUNK_EVENTS
    jobs = [(wl, c) for c in range(n_chunks)]
    if n_chunks > 2:
        with mp.get_context("spawn").Pool(min(n_chunks, max(1, (os.cpu_count() or 2) - 1))) as pool:
            parts = pool.map(_gen_chunk, jobs, chunksize=1)
    else:
        parts = [_gen_chunk(j) for j in jobs]
    u, v = np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts])
    offs, base = [np.zeros(1, np.int64)], 0
    for p in parts:
        offs.append(p[2][1:] + base); base += int(p[2][-1])
    offsets = np.concatenate(offs)[: n_events + 1]
    return np.ascontiguousarray(u[: offsets[-1]]), np.ascontiguousarray(v[: offsets[-1]]), np.ascontiguousarray(offsets)


@pytest.mark.parametrize("cfg,hits_idx,grid_idx,n_sample", [(1, 0, 0, 0), (2, 0, 0, 0), (3, 0, 0, 1500), (4, 1, 2, 1500), (4, 2, 0, 300), (4, 0, 3, 1500)])
def test_full_size_in_the_bench_launch_configuration(cfg, hits_idx, grid_idx, n_sample):
    """Every event of the config at BASELINE.json's size in ONE launch, exactly as bench.py times it (100,000 events of cfg3 on
    the persistent grid: some 675 events per CTA).  Configs 1 and 2 are compared event by event; for cfg3 and the config-4 cells
    the oracle computes a random sample of events one by one (n_found, records, labels), plus two properties that hold at any
    size: every label is -1 or a kept slot, and no event was handed over that the workload's statistics say should not be."""
    wl = synth.workload(cfg, hits_idx, grid_idx)
    u, v, offsets = generate_all(wl, wl.n_events)
    E = wl.n_events
    p = params_of(wl)
    dt = H.HOUGH_U16 if wl.count_dtype == "u16" else H.HOUGH_I32
    g = gpu_run(p, u, v, offsets, dt, want_vote=False)
    assert g["bounds_violations"] == 0 and g["status"] == 0
    if (cfg, hits_idx) != (4, 2):                      # (2000 hits on 128 x 128 switch every bin on: the general kernel's case)
        assert_path(g, fast=True, deferred=0)
    kept = np.minimum(g["n_found"], p.max_candidates)
    lab_event = np.repeat(np.arange(E), np.diff(offsets))
    assert (g["labels"] >= -1).all() and (g["labels"] < kept[lab_event]).all()
    rng = np.random.default_rng(99)
    events = np.arange(E) if n_sample == 0 else np.sort(rng.choice(E, n_sample, replace=False))
    if n_sample == 0:
        o = oracle_run(p, u, v, offsets, want_acc=False)
        np.testing.assert_array_equal(g["n_found"], o["n_found"])
        np.testing.assert_array_equal(g["labels"], o["labels"])
        mask = np.arange(p.max_candidates)[None, :] < np.minimum(o["n_found"], p.max_candidates)[:, None]
        for f in INT_FIELDS + ("theta", "rho"):
            np.testing.assert_array_equal(g["cands"][f][mask], o["cands"][f][mask], err_msg=f)
        return
    for e in events:
        a, z = int(offsets[e]), int(offsets[e + 1])
        o = C.run_batch(u[a:z], v[a:z], np.array([0, z - a], np.int64), p)
        k = min(int(o["n_found"][0]), p.max_candidates)
        assert int(g["n_found"][e]) == int(o["n_found"][0]), e
        assert g["cands"][e, :k].tobytes() == o["cands"][0, :k].tobytes(), e
        np.testing.assert_array_equal(g["labels"][a:z], o["labels"], err_msg=str(e))
