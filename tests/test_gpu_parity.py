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
from util import params_of, std_params

pytestmark = pytest.mark.gpu

INT_FIELDS = ("theta_bin", "rho_bin", "votes", "cluster_root", "cluster_nbins", "reserved")


def make_plan(p: D.Params, n_events, n_hits, max_hpe, count_dtype=H.HOUGH_I32):
    return H.hough_plan_create(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window,
                               p.max_candidates, max(1, n_events), max(0, n_hits), max_hpe, count_dtype,
                               p.hit_frac_bits, p.acc_frac_bits, 0)


def gpu_run(p: D.Params, u, v, offsets, count_dtype=H.HOUGH_I32, want_acc=True, max_hpe=None):
    """Whole CUDA path on one batch; returns numpy results shaped like oracle.hough_c.run_batch."""
    E = len(offsets) - 1
    hpe = int(np.diff(offsets).max()) if E > 0 and len(u) else 0
    plan = make_plan(p, E, len(u), max(hpe, 1) if max_hpe is None else max_hpe, count_dtype)
    du = torch.from_numpy(np.ascontiguousarray(u, np.float32)).cuda()
    dv = torch.from_numpy(np.ascontiguousarray(v, np.float32)).cuda()
    do = torch.from_numpy(np.ascontiguousarray(offsets, np.int64)).cuda()
    out = {}
    acc, dig = H.hough_vote(plan, du, dv, do, want_acc=want_acc, want_digest=True)
    cands, n_found = H.hough_find_clusters(plan, du, dv, do)
    labels = H.hough_assign_hits(plan, du, dv, do, cands, n_found)
    torch.cuda.synchronize()
    out["status"] = H.hough_plan_status(plan)
    if acc is not None:
        a = acc.cpu().numpy()
        out["acc"] = a.view(np.uint16).astype(np.int32) if a.dtype == np.int16 else a
    out["digest"] = dig.cpu().numpy().view(np.uint64)
    out["cands"] = H.candidates_to_numpy(cands)
    out["n_found"] = n_found.cpu().numpy()
    out["labels"] = labels.cpu().numpy()
    out["info"] = H.hough_plan_query(plan)[0]
    H.hough_plan_destroy(plan)
    return out


def assert_same(g, o, p: D.Params, check_acc=True):
    assert g["status"] == 0
    if check_acc and "acc" in g:
        np.testing.assert_array_equal(g["acc"], o["acc"])
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


def oracle_run(p, u, v, offsets):
    return C.run_batch(u, v, offsets, p, want_digest=True, want_acc=True)


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
@pytest.mark.parametrize("cfg,n_events", [(0, 1), (1, 96), (2, 40), (3, 12)])
def test_configs_bit_exact(cfg, n_events):
    wl = synth.workload(cfg)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    dt = H.HOUGH_U16 if wl.count_dtype == "u16" else H.HOUGH_I32
    g = gpu_run(p, b.u, b.v, b.offsets, dt)
    o = oracle_run(p, b.u, b.v, b.offsets)
    assert_same(g, o, p)
    assert g["acc"].sum() == b.n_hits * wl.n_theta     # P4: every generator hit votes once per theta row


@pytest.mark.parametrize("hits_idx,grid_idx,n_events", [(0, 0, 6), (0, 3, 3), (1, 1, 6), (2, 2, 4), (3, 0, 3), (3, 3, 2), (2, 3, 2), (3, 1, 2)])
def test_config4_cells_bit_exact(hits_idx, grid_idx, n_events):
    wl = synth.workload(4, hits_idx, grid_idx)
    b = synth.generate(wl, 0, n_events)
    p = params_of(wl)
    g = gpu_run(p, b.u, b.v, b.offsets)
    o = oracle_run(p, b.u, b.v, b.offsets)
    assert_same(g, o, p)


# ----------------------------------------------------------------------------- adversarial edge set
@pytest.mark.parametrize("case", edge_cases(), ids=lambda c: c[0])
def test_edge_set(case):
    name, p, u, v = case
    offsets = np.array([0, len(u)], np.int64)
    g = gpu_run(p, u, v, offsets, max_hpe=max(len(u), 1))
    o = oracle_run(p, u, v, offsets)
    assert_same(g, o, p)


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


def test_run_host_equals_device_calls():
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 32)
    p = params_of(wl)
    plan = make_plan(p, 32, b.n_hits, int(np.diff(b.offsets).max()))
    cands = np.zeros((32, p.max_candidates, 8), np.int32)
    n_found = np.zeros(32, np.int32)
    labels = np.zeros(b.n_hits, np.int32)
    H.hough_run_host(plan, b.u, b.v, b.offsets, cands, n_found, labels)
    fast = H.hough_plan_query(plan)[0]["fast_groups"] > 0          # fast kernel + general kernel on its deferred list
    assert H.hough_plan_launch_count(plan) == (3 if fast else 2)
    H.hough_plan_destroy(plan)
    o = C.run_batch(b.u, b.v, b.offsets, p)
    np.testing.assert_array_equal(n_found, o["n_found"])
    np.testing.assert_array_equal(labels, o["labels"])
    gc = cands.view(H.CANDIDATE_DTYPE).reshape(32, p.max_candidates)
    for e in range(32):
        k = min(int(n_found[e]), p.max_candidates)
        for f in INT_FIELDS:
            np.testing.assert_array_equal(gc[e, :k][f], o["cands"][e, :k][f])


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
