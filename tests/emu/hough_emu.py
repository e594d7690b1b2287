"""Driver of tests/emu/libhough_emu.so: calls the C ABI of include/hough.h with HOST pointers (the emulated "device").

TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT.  The product binding (paper_2511_02742_b200/hough.py) never loads this
library and has no CPU path; this module exists so that the kernels' logic can be compared with the oracle on a machine
without a GPU (tests/test_emulated_kernels.py).
"""
from __future__ import annotations

import ctypes
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

CAND_DTYPE = np.dtype([("theta_bin", "<i4"), ("rho_bin", "<i4"), ("votes", "<i4"), ("cluster_root", "<i4"),
                       ("cluster_nbins", "<i4"), ("theta", "<f4"), ("rho", "<f4"), ("reserved", "<i4")])
HOUGH_I32, HOUGH_U16 = 0, 1
FLAG_GENERAL_ONLY, FLAG_SMALL_LISTS, FLAG_THETA_WRAP = 1, 2, 4


class Desc(ctypes.Structure):
    _fields_ = [("n_theta", ctypes.c_int32), ("n_rho", ctypes.c_int32), ("rho_min", ctypes.c_double),
                ("rho_max", ctypes.c_double), ("coord_max", ctypes.c_double), ("hit_frac_bits", ctypes.c_int32),
                ("acc_frac_bits", ctypes.c_int32), ("vote_threshold", ctypes.c_int32), ("assign_window", ctypes.c_double),
                ("max_candidates", ctypes.c_int32), ("count_dtype", ctypes.c_int32), ("max_events", ctypes.c_int32),
                ("max_hits", ctypes.c_int64), ("max_hits_per_event", ctypes.c_int32), ("flags", ctypes.c_int32),
                ("device", ctypes.c_int32), ("theta_min", ctypes.c_double), ("theta_max", ctypes.c_double)]


INFO_FIELDS = ("hit_frac_bits", "acc_frac_bits", "rho_offset_q", "assign_window_q", "strip_rows", "n_strips", "counter_bytes",
               "threads_per_cta", "ctas_per_sm", "n_ctas", "smem_bytes_per_cta", "n_sm", "fast_groups", "fast_threads",
               "fast_ctas", "fast_smem_bytes", "fast_hits_cap", "fast_on_cap", "fast_peak_cap", "fast_strip_list_cap")


class Info(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in INFO_FIELDS]


_lib = None


def lib():
    global _lib
    if _lib is None:
        spec = importlib.util.spec_from_file_location("build_emu", os.path.join(_HERE, "build_emu.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        # HOUGH_EMU_LIB=tsan: the race-detector build (the process must have been started with libtsan preloaded: race_check.py);
        # HOUGH_EMU_LIB=/path/to.so: a library race_check.py --self-test built
        which = os.environ.get("HOUGH_EMU_LIB", "")
        L = ctypes.CDLL(mod.build_tsan() if which == "tsan" else (which if which else mod.build()))
        vp, i32 = ctypes.c_void_p, ctypes.c_int32
        L.hough_plan_create.argtypes = [ctypes.POINTER(Desc), ctypes.POINTER(vp)]
        L.hough_plan_destroy.argtypes = [vp]
        L.hough_vote.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
        L.hough_find_clusters.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
        L.hough_assign_hits.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp, vp]
        L.hough_run_host_chunked.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp, i32]
        L.hough_plan_query.argtypes = [vp, ctypes.POINTER(Info), vp, vp]
        L.hough_plan_status.argtypes = [vp, ctypes.POINTER(i32), vp]
        L.hough_plan_debug_counters.argtypes = [vp, vp, vp]
        L.hough_plan_launch_count.argtypes = [vp]
        L.hough_plan_launch_count.restype = ctypes.c_int64
        L.cuda_emu_violations.restype = ctypes.c_longlong
        L.cuda_emu_first_violation.restype = ctypes.c_char_p
        L.cuda_emu_configure.argtypes = [ctypes.c_ulonglong, ctypes.c_int, ctypes.c_uint]
        _lib = L
    return _lib


def configure(seed: int = 0, preempt_per_1024: int = 0, smem_window: int = 1024, workers: int = 1):
    """Schedule seed, chance of a switch at every atomic / cache-bypassing access, shared-window address of the dynamic
    shared memory (what cvta.to.shared returns for its first byte), CTAs of a grid that run at the same time (each on its
    own OS thread; 1 = one after another)."""
    lib().cuda_emu_configure(seed, preempt_per_1024, smem_window)
    lib().cuda_emu_set_workers(workers)


def theta_window(p):
    """(theta_min, theta_max) of the descriptor for oracle parameters: the default window is spelled (0, 0)."""
    import math
    lo, hi = getattr(p, "theta_min", 0.0), getattr(p, "theta_max", math.pi)
    return (0.0, 0.0) if (lo == 0.0 and hi == math.pi) else (lo, hi)


class DevBuf:
    """A "device" buffer of the emulated runtime is plain host memory; inputs are copied so that alignment is the caller's."""

    def __init__(self, a: np.ndarray):
        self.a = np.ascontiguousarray(a)
        # 16-byte aligned storage (the ABI asks for it)
        raw = np.empty(self.a.nbytes + 32, np.uint8)
        off = (-raw.ctypes.data) % 16
        self.raw = raw
        self.view = raw[off:off + self.a.nbytes].view(self.a.dtype).reshape(self.a.shape)
        self.view[...] = self.a

    @property
    def ptr(self):
        return ctypes.c_void_p(self.view.ctypes.data) if self.view.size else ctypes.c_void_p(self.raw.ctypes.data + (-self.raw.ctypes.data) % 16)


def run(p, u, v, offsets, count_dtype=HOUGH_I32, want_acc=True, max_hpe=None, flags=0, want_vote=True):
    """The whole path through the C ABI on the emulated device; same result dict as tests/test_gpu_parity.gpu_run."""
    L = lib()
    L.cuda_emu_reset_violations()
    E = len(offsets) - 1
    hpe = int(np.diff(offsets).max()) if E > 0 and len(u) else 0
    if getattr(p, "theta_wrap", False):
        flags |= FLAG_THETA_WRAP
    d = Desc(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.hit_frac_bits, p.acc_frac_bits, p.vote_threshold,
             p.assign_window, p.max_candidates, count_dtype, max(1, E), max(0, len(u)), max(hpe, 1) if max_hpe is None else max_hpe,
             flags, 0, *theta_window(p))
    h = ctypes.c_void_p()
    rc = L.hough_plan_create(ctypes.byref(d), ctypes.byref(h))
    assert rc == 0, f"hough_plan_create -> {rc}"
    du, dv = DevBuf(np.asarray(u, np.float32)), DevBuf(np.asarray(v, np.float32))
    do = DevBuf(np.asarray(offsets, np.int64))
    out = {}
    K = p.max_candidates
    if want_vote:
        acc = DevBuf(np.zeros((E, p.n_theta, p.n_rho), np.uint16 if count_dtype == HOUGH_U16 else np.int32)) if want_acc else None
        dig = DevBuf(np.zeros(E, np.uint64))
        rc = L.hough_vote(h, du.ptr, dv.ptr, do.ptr, E, acc.ptr if acc else None, dig.ptr, None)
        assert rc == 0, f"hough_vote -> {rc}"
        if acc:
            out["acc"] = acc.view.astype(np.int32)
        out["digest"] = dig.view.copy()
    cands = DevBuf(np.zeros((E, K), CAND_DTYPE))
    n_found = DevBuf(np.zeros(E, np.int32))
    labels = DevBuf(np.full(len(u), -99, np.int32))
    rc = L.hough_find_clusters(h, du.ptr, dv.ptr, do.ptr, E, cands.ptr, n_found.ptr, None)
    assert rc == 0, f"hough_find_clusters -> {rc}"
    rc = L.hough_assign_hits(h, du.ptr, dv.ptr, do.ptr, E, cands.ptr, n_found.ptr, labels.ptr, None)
    assert rc == 0, f"hough_assign_hits -> {rc}"
    dbg = np.zeros(16, np.uint64)
    L.hough_plan_debug_counters(h, dbg.ctypes.data, None)
    st = ctypes.c_int32(0)
    L.hough_plan_status(h, ctypes.byref(st), None)
    info = Info()
    L.hough_plan_query(h, ctypes.byref(info), None, None)
    out.update(status=st.value, deferred=int(dbg[15]), bounds_violations=int(dbg[14]), bounds_site=int(dbg[13]),
               cands=cands.view.copy(), n_found=n_found.view.copy(), labels=labels.view.copy(),
               info={n: getattr(info, n) for n in INFO_FIELDS}, launches=int(L.hough_plan_launch_count(h)),
               emu_violations=int(L.cuda_emu_violations()), emu_first_violation=L.cuda_emu_first_violation().decode())
    L.hough_plan_destroy(h)
    return out


def assign(p, u, v, offsets, cands, n_found, count_dtype=HOUGH_I32):
    """hough_assign_hits alone, on caller-made records (cands [E][K] of CAND_DTYPE, n_found [E]) -> (labels, return code)."""
    L = lib()
    L.cuda_emu_reset_violations()
    E = len(offsets) - 1
    hpe = int(np.diff(offsets).max()) if E > 0 and len(u) else 0
    d = Desc(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.hit_frac_bits, p.acc_frac_bits, p.vote_threshold,
             p.assign_window, p.max_candidates, count_dtype, max(1, E), max(0, len(u)), max(hpe, 1), 0, 0, *theta_window(p))
    h = ctypes.c_void_p()
    assert L.hough_plan_create(ctypes.byref(d), ctypes.byref(h)) == 0
    du, dv, do = DevBuf(np.asarray(u, np.float32)), DevBuf(np.asarray(v, np.float32)), DevBuf(np.asarray(offsets, np.int64))
    dc, dn = DevBuf(np.ascontiguousarray(cands, CAND_DTYPE)), DevBuf(np.asarray(n_found, np.int32))
    labels = DevBuf(np.full(len(u), -99, np.int32))
    rc = L.hough_assign_hits(h, du.ptr, dv.ptr, do.ptr, E, dc.ptr, dn.ptr, labels.ptr, None)
    rc_null = L.hough_assign_hits(h, du.ptr, dv.ptr, do.ptr, E, dc.ptr, dn.ptr, None, None)
    dbg = np.zeros(16, np.uint64)
    L.hough_plan_debug_counters(h, dbg.ctypes.data, None)
    L.hough_plan_destroy(h)
    assert L.cuda_emu_violations() == 0, L.cuda_emu_first_violation().decode()
    assert int(dbg[14]) == 0, f"index check failed at site {int(dbg[13])}"
    return labels.view.copy(), rc, rc_null


def run_host(p, u, v, offsets, n_chunks, count_dtype=HOUGH_I32, repeat=1):
    """hough_run_host_chunked on the emulated device (called `repeat` times on one plan; the last results are returned)."""
    L = lib()
    L.cuda_emu_reset_violations()
    E = len(offsets) - 1
    hpe = int(np.diff(offsets).max()) if E > 0 and len(u) else 0
    d = Desc(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.hit_frac_bits, p.acc_frac_bits, p.vote_threshold,
             p.assign_window, p.max_candidates, count_dtype, max(1, E), max(0, len(u)), max(hpe, 1), 0, 0)
    h = ctypes.c_void_p()
    assert L.hough_plan_create(ctypes.byref(d), ctypes.byref(h)) == 0
    u, v = np.ascontiguousarray(u, np.float32), np.ascontiguousarray(v, np.float32)
    offsets = np.ascontiguousarray(offsets, np.int64)
    for _ in range(repeat):
        cands = np.zeros((E, p.max_candidates), CAND_DTYPE)
        n_found = np.full(E, -7, np.int32)
        labels = np.full(len(u), -7, np.int32)
        rc = L.hough_run_host_chunked(h, u.ctypes.data, v.ctypes.data, offsets.ctypes.data, E, cands.ctypes.data,
                                      n_found.ctypes.data, labels.ctypes.data, n_chunks)
        assert rc == 0, f"hough_run_host_chunked -> {rc}"
    out = dict(cands=cands, n_found=n_found, labels=labels, launches=int(L.hough_plan_launch_count(h)),
               emu_violations=int(L.cuda_emu_violations()), emu_first_violation=L.cuda_emu_first_violation().decode())
    L.hough_plan_destroy(h)
    return out


# ----------------------------------------------------------------------------- stages around the core
FIT_DTYPE = np.dtype([("n_hits", "<i4"), ("max_run", "<i4"), ("plane_mask", "<u8"), ("slope", "<f4"), ("intercept", "<f4"),
                      ("flags", "<i4"), ("reserved", "<i4")])
assert FIT_DTYPE.itemsize == 32


class PlaneGeometry(ctypes.Structure):
    _fields_ = [("plane_origin", ctypes.c_double), ("plane_pitch", ctypes.c_double), ("n_planes", ctypes.c_int32),
                ("min_run", ctypes.c_int32), ("wrap", ctypes.c_int32), ("reserved", ctypes.c_int32)]


class FrontDesc(ctypes.Structure):
    _fields_ = [("t0", ctypes.c_double), ("window_width", ctypes.c_double), ("window_step", ctypes.c_double),
                ("windows_per_fill", ctypes.c_int32), ("xy_max", ctypes.c_double), ("max_fills", ctypes.c_int32),
                ("max_hits", ctypes.c_int64), ("device", ctypes.c_int32), ("reserved", ctypes.c_int32)]


def refit(p, u, v, offsets, n_found, labels, geom, count_dtype=HOUGH_I32, max_hpe=None):
    """hough_refit_tracks on the emulated device -> (fits [E][K] structured array, return code)."""
    L = lib()
    L.cuda_emu_reset_violations()
    vp, i32 = ctypes.c_void_p, ctypes.c_int32
    L.hough_refit_tracks.argtypes = [vp, vp, vp, vp, i32, vp, vp, ctypes.POINTER(PlaneGeometry), vp, vp]
    E = len(offsets) - 1
    hpe = int(np.diff(offsets).max()) if E > 0 and len(u) else 0
    d = Desc(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.hit_frac_bits, p.acc_frac_bits, p.vote_threshold,
             p.assign_window, p.max_candidates, count_dtype, max(1, E), max(0, len(u)), max(hpe, 1) if max_hpe is None else max_hpe, 0, 0)
    h = ctypes.c_void_p()
    assert L.hough_plan_create(ctypes.byref(d), ctypes.byref(h)) == 0
    du, dv, do = DevBuf(np.asarray(u, np.float32)), DevBuf(np.asarray(v, np.float32)), DevBuf(np.asarray(offsets, np.int64))
    dn, dl = DevBuf(np.asarray(n_found, np.int32)), DevBuf(np.asarray(labels, np.int32))
    fits = DevBuf(np.zeros((E, p.max_candidates), FIT_DTYPE))
    g = PlaneGeometry(geom.origin, geom.pitch, geom.n_planes, geom.min_run, int(geom.wrap), 0)
    rc = L.hough_refit_tracks(h, du.ptr, dv.ptr, do.ptr, E, dn.ptr, dl.ptr, ctypes.byref(g), fits.ptr, None)
    dbg = np.zeros(16, np.uint64)
    L.hough_plan_debug_counters(h, dbg.ctypes.data, None)
    L.hough_plan_destroy(h)
    assert L.cuda_emu_violations() == 0, L.cuda_emu_first_violation().decode()
    assert int(dbg[14]) == 0, f"index check failed at site {int(dbg[13])}"
    return fits.view.copy(), rc


def frontend_slice(fe, x, y, z, t, fill_offsets, capacity=None):
    """hough_frontend_* on the emulated device.  fe: oracle.track_def.FrontEnd (field names only; no arithmetic is shared).
    -> dict(u, v, src, offsets, status)"""
    L = lib()
    L.cuda_emu_reset_violations()
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    L.hough_frontend_create.argtypes = [ctypes.POINTER(FrontDesc), ctypes.POINTER(vp)]
    L.hough_frontend_destroy.argtypes = [vp]
    L.hough_frontend_slice.argtypes = [vp, vp, vp, vp, vp, vp, i32, i64, vp, vp, vp, vp, i64, vp]
    L.hough_frontend_status.argtypes = [vp, ctypes.POINTER(i32), vp]
    n_fills, n = len(fill_offsets) - 1, len(x)
    d = FrontDesc(fe.t0, fe.width, fe.step, fe.windows_per_fill, fe.xy_max, max(1, n_fills), n, 0, 0)
    h = vp()
    rc = L.hough_frontend_create(ctypes.byref(d), ctypes.byref(h))
    assert rc == 0, f"hough_frontend_create -> {rc}"
    m = -(-int(round(fe.width * 256)) // int(round(fe.step * 256)))
    cap = m * n if capacity is None else capacity
    bx, by, bz, bt = (DevBuf(np.asarray(a, np.float32)) for a in (x, y, z, t))
    bf = DevBuf(np.asarray(fill_offsets, np.int64))
    bu, bv = DevBuf(np.full(cap, np.nan, np.float32)), DevBuf(np.full(cap, np.nan, np.float32))
    bs = DevBuf(np.full(cap, -1, np.int32))
    bo = DevBuf(np.full(n_fills * fe.windows_per_fill + 1, -1, np.int64))
    rc = L.hough_frontend_slice(h, bx.ptr, by.ptr, bz.ptr, bt.ptr, bf.ptr, n_fills, n, bu.ptr, bv.ptr, bs.ptr, bo.ptr, cap, None)
    assert rc == 0, f"hough_frontend_slice -> {rc}"
    st = i32(0)
    L.hough_frontend_status(h, ctypes.byref(st), None)
    L.hough_frontend_destroy(h)
    assert L.cuda_emu_violations() == 0, L.cuda_emu_first_violation().decode()
    return dict(u=bu.view.copy(), v=bv.view.copy(), src=bs.view.copy(), offsets=bo.view.copy(), status=st.value)


def peeloff(p, u, v, offsets, max_hpe=None):
    """hough_find_tracks_peeloff on the emulated device -> dict(cands, n_found, labels, status)."""
    L = lib()
    L.cuda_emu_reset_violations()
    vp, i32 = ctypes.c_void_p, ctypes.c_int32
    L.hough_find_tracks_peeloff.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp, vp]
    E = len(offsets) - 1
    hpe = int(np.diff(offsets).max()) if E > 0 and len(u) else 0
    d = Desc(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.hit_frac_bits, p.acc_frac_bits, p.vote_threshold,
             p.assign_window, p.max_candidates, HOUGH_I32, max(1, E), max(0, len(u)), max(hpe, 1) if max_hpe is None else max_hpe, 0, 0)
    h = ctypes.c_void_p()
    assert L.hough_plan_create(ctypes.byref(d), ctypes.byref(h)) == 0
    du, dv, do = DevBuf(np.asarray(u, np.float32)), DevBuf(np.asarray(v, np.float32)), DevBuf(np.asarray(offsets, np.int64))
    cands = DevBuf(np.zeros((E, p.max_candidates), CAND_DTYPE))
    n_found = DevBuf(np.full(E, -5, np.int32))
    labels = DevBuf(np.full(max(len(u), 1), -99, np.int32))
    rc = L.hough_find_tracks_peeloff(h, du.ptr, dv.ptr, do.ptr, E, cands.ptr, n_found.ptr, labels.ptr, None)
    assert rc == 0, f"hough_find_tracks_peeloff -> {rc}"
    dbg = np.zeros(16, np.uint64)
    L.hough_plan_debug_counters(h, dbg.ctypes.data, None)
    st = ctypes.c_int32(0)
    L.hough_plan_status(h, ctypes.byref(st), None)
    L.hough_plan_destroy(h)
    assert L.cuda_emu_violations() == 0, L.cuda_emu_first_violation().decode()
    assert int(dbg[14]) == 0, f"index check failed at site {int(dbg[13])}"
    return dict(cands=cands.view.copy(), n_found=n_found.view.copy(), labels=labels.view[: len(u)].copy(), status=st.value)


def two_stage(p, u, v, offsets, c_theta, c_rho):
    """hough_find_two_stage on the emulated device -> dict(cands, n_found, rc)."""
    L = lib()
    L.cuda_emu_reset_violations()
    vp, i32 = ctypes.c_void_p, ctypes.c_int32
    L.hough_find_two_stage.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, vp]
    E = len(offsets) - 1
    hpe = int(np.diff(offsets).max()) if E > 0 and len(u) else 0
    d = Desc(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.hit_frac_bits, p.acc_frac_bits, p.vote_threshold,
             p.assign_window, p.max_candidates, HOUGH_I32, max(1, E), max(0, len(u)), max(hpe, 1), 0, 0)
    h = ctypes.c_void_p()
    assert L.hough_plan_create(ctypes.byref(d), ctypes.byref(h)) == 0
    du, dv, do = DevBuf(np.asarray(u, np.float32)), DevBuf(np.asarray(v, np.float32)), DevBuf(np.asarray(offsets, np.int64))
    cands = DevBuf(np.zeros((E, p.max_candidates), CAND_DTYPE))
    n_found = DevBuf(np.full(E, -5, np.int32))
    rc = L.hough_find_two_stage(h, du.ptr, dv.ptr, do.ptr, E, c_theta, c_rho, cands.ptr, n_found.ptr, None)
    dbg = np.zeros(16, np.uint64)
    L.hough_plan_debug_counters(h, dbg.ctypes.data, None)
    L.hough_plan_destroy(h)
    assert L.cuda_emu_violations() == 0, L.cuda_emu_first_violation().decode()
    assert int(dbg[14]) == 0, f"index check failed at site {int(dbg[13])}"
    return dict(cands=cands.view.copy(), n_found=n_found.view.copy(), rc=rc)
