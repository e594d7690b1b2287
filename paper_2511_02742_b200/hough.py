"""Thin ctypes binding of libhough.so -- the same names as include/hough.h, argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; torch is used for device memory and streams.
There is no CPU fallback: if the shared library is missing or fails to load, importing the entry points raises.

    plan = hough_plan_create(n_theta=512, n_rho=512, rho_min=-256, rho_max=256, coord_max=256, vote_threshold=20,
                             assign_window=1.0, max_candidates=128, max_events=E, max_hits=N, max_hits_per_event=4096)
    cands, n_found = hough_find_clusters(plan, u, v, offsets)        # torch CUDA tensors in, torch CUDA tensors out
    labels = hough_assign_hits(plan, u, v, offsets, cands, n_found)
    hough_plan_destroy(plan)
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhough.so")

HOUGH_OK, HOUGH_EINVAL, HOUGH_ERANGE, HOUGH_ECUDA, HOUGH_ENOMEM = 0, -1, -2, -3, -4
HOUGH_I32, HOUGH_U16 = 0, 1
HOUGH_STATUS_EVENT_TOO_LONG, HOUGH_STATUS_BAD_OFFSETS, HOUGH_STATUS_INTERNAL = 1, 2, 4
HOUGH_FLAG_GENERAL_ONLY, HOUGH_FLAG_SMALL_LISTS, HOUGH_FLAG_THETA_WRAP = 1, 2, 4

# numpy view of hough_candidate_t (32 bytes)
CANDIDATE_DTYPE = np.dtype([("theta_bin", "<i4"), ("rho_bin", "<i4"), ("votes", "<i4"), ("cluster_root", "<i4"),
                            ("cluster_nbins", "<i4"), ("theta", "<f4"), ("rho", "<f4"), ("reserved", "<i4")])
CANDIDATE_WORDS = 8   # a record is 8 x 32-bit words; device tensors of records are int32 [E, K, 8]

EXPORTS = ("hough_plan_create", "hough_plan_destroy", "hough_vote", "hough_find_clusters", "hough_assign_hits",
           "hough_run_host", "hough_run_host_chunked", "hough_plan_query", "hough_plan_status", "hough_plan_launch_count", "hough_plan_debug_counters",
           "hough_measure_smem_atomic_peak", "hough_strerror", "hough_last_cuda_error", "hough_version",
           "hough_refit_tracks", "hough_frontend_create", "hough_frontend_destroy", "hough_frontend_slice",
           "hough_frontend_status", "hough_find_tracks_peeloff", "hough_find_two_stage")


class hough_plan_desc_t(ctypes.Structure):
    _fields_ = [("n_theta", ctypes.c_int32), ("n_rho", ctypes.c_int32), ("rho_min", ctypes.c_double),
                ("rho_max", ctypes.c_double), ("coord_max", ctypes.c_double), ("hit_frac_bits", ctypes.c_int32),
                ("acc_frac_bits", ctypes.c_int32), ("vote_threshold", ctypes.c_int32), ("assign_window", ctypes.c_double),
                ("max_candidates", ctypes.c_int32), ("count_dtype", ctypes.c_int32), ("max_events", ctypes.c_int32),
                ("max_hits", ctypes.c_int64), ("max_hits_per_event", ctypes.c_int32), ("flags", ctypes.c_int32),
                ("device", ctypes.c_int32), ("theta_min", ctypes.c_double), ("theta_max", ctypes.c_double)]


class hough_plan_info_t(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("hit_frac_bits", "acc_frac_bits", "rho_offset_q", "assign_window_q",
                                              "strip_rows", "n_strips", "counter_bytes", "threads_per_cta", "ctas_per_sm",
                                              "n_ctas", "smem_bytes_per_cta", "n_sm", "fast_groups", "fast_threads",
                                              "fast_ctas", "fast_smem_bytes", "fast_hits_cap", "fast_on_cap", "fast_peak_cap",
                                              "fast_strip_list_cap")]


# numpy view of hough_fit_t (32 bytes); device tensors of fit records are int32 [E, K, 8]
FIT_DTYPE = np.dtype([("n_hits", "<i4"), ("max_run", "<i4"), ("plane_mask", "<u8"), ("slope", "<f4"), ("intercept", "<f4"),
                      ("flags", "<i4"), ("reserved", "<i4")])
HOUGH_FIT_FOUND, HOUGH_FIT_DEGENERATE = 1, 2
HOUGH_STATUS_OUTPUT_TRUNCATED = 8


class hough_plane_geometry_t(ctypes.Structure):
    _fields_ = [("plane_origin", ctypes.c_double), ("plane_pitch", ctypes.c_double), ("n_planes", ctypes.c_int32),
                ("min_run", ctypes.c_int32), ("wrap", ctypes.c_int32), ("reserved", ctypes.c_int32)]


class hough_frontend_desc_t(ctypes.Structure):
    _fields_ = [("t0", ctypes.c_double), ("window_width", ctypes.c_double), ("window_step", ctypes.c_double),
                ("windows_per_fill", ctypes.c_int32), ("xy_max", ctypes.c_double), ("max_fills", ctypes.c_int32),
                ("max_hits", ctypes.c_int64), ("device", ctypes.c_int32), ("reserved", ctypes.c_int32)]


class HoughError(RuntimeError):
    def __init__(self, status: int, where: str):
        lib = _lib
        msg = lib.hough_strerror(status).decode() if lib is not None else "?"
        cuda = lib.hough_last_cuda_error().decode() if (lib is not None and status == HOUGH_ECUDA) else ""
        super().__init__(f"{where}: {msg} ({status})" + (f" [{cuda}]" if cuda else ""))
        self.status = status


_lib = None


def load_library(path: Optional[str] = None) -> ctypes.CDLL:
    """dlopen libhough.so and declare the prototypes of include/hough.h.  Raises if the library is not built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_2511_02742_b200.build` "
                           "(there is no CPU fallback for the Hough kernels)")
    L = ctypes.CDLL(path)
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    L.hough_plan_create.argtypes = [ctypes.POINTER(hough_plan_desc_t), ctypes.POINTER(vp)]
    L.hough_plan_destroy.argtypes = [vp]
    L.hough_vote.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
    L.hough_find_clusters.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
    L.hough_assign_hits.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp, vp]
    L.hough_run_host.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
    L.hough_run_host_chunked.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp, i32]
    L.hough_plan_query.argtypes = [vp, ctypes.POINTER(hough_plan_info_t), vp, vp]
    L.hough_plan_status.argtypes = [vp, ctypes.POINTER(i32), vp]
    L.hough_plan_launch_count.argtypes = [vp]
    L.hough_plan_launch_count.restype = i64
    L.hough_plan_debug_counters.argtypes = [vp, vp, vp]
    L.hough_measure_smem_atomic_peak.argtypes = [i32, ctypes.c_double, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.hough_strerror.argtypes = [ctypes.c_int]
    L.hough_strerror.restype = ctypes.c_char_p
    L.hough_last_cuda_error.argtypes = []
    L.hough_last_cuda_error.restype = ctypes.c_char_p
    L.hough_version.argtypes = []
    L.hough_refit_tracks.argtypes = [vp, vp, vp, vp, i32, vp, vp, ctypes.POINTER(hough_plane_geometry_t), vp, vp]
    L.hough_find_tracks_peeloff.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp, vp]
    L.hough_find_two_stage.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, vp]
    L.hough_frontend_create.argtypes = [ctypes.POINTER(hough_frontend_desc_t), ctypes.POINTER(vp)]
    L.hough_frontend_destroy.argtypes = [vp]
    L.hough_frontend_slice.argtypes = [vp, vp, vp, vp, vp, vp, i32, i64, vp, vp, vp, vp, i64, vp]
    L.hough_frontend_status.argtypes = [vp, ctypes.POINTER(i32), vp]
    for name in EXPORTS:
        if name not in ("hough_strerror", "hough_last_cuda_error", "hough_plan_launch_count"):
            getattr(L, name).restype = ctypes.c_int
    _lib = L
    return L


def _check(status: int, where: str):
    if status != HOUGH_OK:
        raise HoughError(status, where)


class Plan:
    """Owner of a hough_plan_t* (opaque handle) plus the descriptor it was made from."""

    def __init__(self, handle: int, desc: hough_plan_desc_t):
        self.handle = ctypes.c_void_p(handle)
        self.desc = desc
        self.n_theta, self.n_rho, self.K = desc.n_theta, desc.n_rho, desc.max_candidates
        self.device = torch.device("cuda", desc.device)

    def __del__(self):
        try:
            hough_plan_destroy(self)
        except Exception:
            pass


def hough_plan_create(n_theta: int, n_rho: int, rho_min: float, rho_max: float, coord_max: float, vote_threshold: int,
                      assign_window: float, max_candidates: int, max_events: int, max_hits: int, max_hits_per_event: int,
                      count_dtype: int = HOUGH_I32, hit_frac_bits: int = -1, acc_frac_bits: int = -1, device: int = 0,
                      flags: int = 0, theta_min: float = 0.0, theta_max: float = 0.0) -> Plan:
    L = load_library()
    d = hough_plan_desc_t(n_theta, n_rho, rho_min, rho_max, coord_max, hit_frac_bits, acc_frac_bits, vote_threshold,
                          assign_window, max_candidates, count_dtype, max_events, max_hits, max_hits_per_event, flags, device,
                          theta_min, theta_max)
    h = ctypes.c_void_p()
    _check(L.hough_plan_create(ctypes.byref(d), ctypes.byref(h)), "hough_plan_create")
    return Plan(h.value, d)


def hough_plan_destroy(plan: Plan) -> None:
    if plan.handle is not None and plan.handle.value:
        h, plan.handle = plan.handle, None
        _check(load_library().hough_plan_destroy(h), "hough_plan_destroy")


def hough_plan_query(plan: Plan) -> Tuple[dict, np.ndarray, np.ndarray]:
    """(info dict, C_q int32 [n_theta], S_q int32 [n_theta])."""
    info = hough_plan_info_t()
    c = np.zeros(plan.n_theta, np.int32)
    s = np.zeros(plan.n_theta, np.int32)
    _check(load_library().hough_plan_query(plan.handle, ctypes.byref(info), c.ctypes.data, s.ctypes.data), "hough_plan_query")
    return {n: getattr(info, n) for n, _ in hough_plan_info_t._fields_}, c, s


def hough_plan_status(plan: Plan, stream: Optional[torch.cuda.Stream] = None) -> int:
    out = ctypes.c_int32(0)
    _check(load_library().hough_plan_status(plan.handle, ctypes.byref(out), _stream_ptr(plan, stream)), "hough_plan_status")
    return out.value


def hough_plan_launch_count(plan: Plan) -> int:
    return int(load_library().hough_plan_launch_count(plan.handle))


def hough_plan_debug_counters(plan: Plan, stream=None) -> np.ndarray:
    """uint64 [16]: per-phase SM-cycle sums (zeros unless libhough was built with -DHOUGH_PHASE_TIMERS; cleared);
    [15] = events the last hough_find_clusters call deferred from the fast to the general kernel; [14], [13] = failed
    index checks and the first failing site (only the -DHOUGH_BOUNDS build can report non-zero)."""
    out = np.zeros(16, np.uint64)
    _check(load_library().hough_plan_debug_counters(plan.handle, out.ctypes.data, _stream_ptr(plan, stream)),
           "hough_plan_debug_counters")
    return out


def _stream_ptr(plan: Plan, stream) -> ctypes.c_void_p:
    s = stream if stream is not None else torch.cuda.current_stream(plan.device)
    return ctypes.c_void_p(s.cuda_stream)


def _dev(plan: Plan, t: torch.Tensor, dtype: torch.dtype, name: str) -> ctypes.c_void_p:
    if t.dtype != dtype or not t.is_cuda or t.device != plan.device or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous {dtype} tensor on {plan.device}, got {t.dtype} on {t.device}")
    return ctypes.c_void_p(t.data_ptr())


def _n_events(offsets: torch.Tensor) -> int:
    if offsets.dim() != 1 or offsets.numel() < 1:
        raise ValueError("offsets must be a 1-D tensor of n_events + 1 entries")
    return offsets.numel() - 1


def hough_vote(plan: Plan, u: torch.Tensor, v: torch.Tensor, offsets: torch.Tensor, want_acc: bool = True,
               want_digest: bool = False, stream=None) -> Tuple[Optional[torch.Tensor], Optional[torch.Tensor]]:
    """(acc [E, n_theta, n_rho] int32 or int16-as-uint16 bits, digest [E] int64-as-uint64 bits); either may be None."""
    E = _n_events(offsets)
    acc = dig = None
    if want_acc:
        dt = torch.int16 if plan.desc.count_dtype == HOUGH_U16 else torch.int32
        acc = torch.empty((E, plan.n_theta, plan.n_rho), dtype=dt, device=plan.device)
    if want_digest:
        dig = torch.empty(E, dtype=torch.int64, device=plan.device)
    _check(load_library().hough_vote(plan.handle, _dev(plan, u, torch.float32, "u"), _dev(plan, v, torch.float32, "v"),
                                     _dev(plan, offsets, torch.int64, "offsets"), E,
                                     None if acc is None else ctypes.c_void_p(acc.data_ptr()),
                                     None if dig is None else ctypes.c_void_p(dig.data_ptr()), _stream_ptr(plan, stream)),
           "hough_vote")
    return acc, dig


def hough_find_clusters(plan: Plan, u: torch.Tensor, v: torch.Tensor, offsets: torch.Tensor,
                        cands: Optional[torch.Tensor] = None, n_found: Optional[torch.Tensor] = None, stream=None):
    """(cands int32 [E, K, 8] -- the 32-byte records as words, n_found int32 [E]).  Rows beyond min(n_found, K) are untouched."""
    E = _n_events(offsets)
    if cands is None:
        cands = torch.zeros((E, plan.K, CANDIDATE_WORDS), dtype=torch.int32, device=plan.device)
    if n_found is None:
        n_found = torch.zeros(E, dtype=torch.int32, device=plan.device)
    _check(load_library().hough_find_clusters(plan.handle, _dev(plan, u, torch.float32, "u"), _dev(plan, v, torch.float32, "v"),
                                              _dev(plan, offsets, torch.int64, "offsets"), E,
                                              _dev(plan, cands, torch.int32, "cands"), _dev(plan, n_found, torch.int32, "n_found"),
                                              _stream_ptr(plan, stream)), "hough_find_clusters")
    return cands, n_found


def hough_assign_hits(plan: Plan, u: torch.Tensor, v: torch.Tensor, offsets: torch.Tensor, cands: torch.Tensor,
                      n_found: torch.Tensor, labels: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """labels int32 [N]."""
    E = _n_events(offsets)
    if labels is None:
        labels = torch.empty(u.numel(), dtype=torch.int32, device=plan.device)
    _check(load_library().hough_assign_hits(plan.handle, _dev(plan, u, torch.float32, "u"), _dev(plan, v, torch.float32, "v"),
                                            _dev(plan, offsets, torch.int64, "offsets"), E,
                                            _dev(plan, cands, torch.int32, "cands"), _dev(plan, n_found, torch.int32, "n_found"),
                                            _dev(plan, labels, torch.int32, "labels"), _stream_ptr(plan, stream)),
           "hough_assign_hits")
    return labels


def _host(t, dtype, name):
    if isinstance(t, np.ndarray):
        if t.dtype != dtype or not t.flags.c_contiguous:
            raise TypeError(f"{name}: expected a C-contiguous {dtype} array")
        return ctypes.c_void_p(t.ctypes.data)
    if t.is_cuda or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous host tensor")
    return ctypes.c_void_p(t.data_ptr())


def hough_run_host(plan: Plan, u, v, offsets, cands, n_found, labels, n_chunks: int = 0) -> None:
    """Whole pipeline on HOST buffers (numpy arrays or CPU torch tensors, ideally pinned); outputs are filled in place.
    cands: int32 [E, K, 8] (or CANDIDATE_DTYPE [E, K]); n_found int32 [E]; labels int32 [N]; any output may be None.
    n_chunks > 0 calls hough_run_host_chunked with that many chunks."""
    E = int(offsets.shape[0]) - 1
    if n_chunks:
        return hough_run_host_chunked(plan, u, v, offsets, cands, n_found, labels, n_chunks)
    _check(load_library().hough_run_host(plan.handle, _host(u, np.float32, "u"), _host(v, np.float32, "v"),
                                         _host(offsets, np.int64, "offsets"), E,
                                         None if cands is None else ctypes.c_void_p(cands.ctypes.data if isinstance(cands, np.ndarray) else cands.data_ptr()),
                                         None if n_found is None else _host(n_found, np.int32, "n_found"),
                                         None if labels is None else _host(labels, np.int32, "labels")), "hough_run_host")


def hough_run_host_chunked(plan: Plan, u, v, offsets, cands, n_found, labels, n_chunks: int) -> None:
    E = int(offsets.shape[0]) - 1
    _check(load_library().hough_run_host_chunked(
        plan.handle, _host(u, np.float32, "u"), _host(v, np.float32, "v"), _host(offsets, np.int64, "offsets"), E,
        None if cands is None else ctypes.c_void_p(cands.ctypes.data if isinstance(cands, np.ndarray) else cands.data_ptr()),
        None if n_found is None else _host(n_found, np.int32, "n_found"),
        None if labels is None else _host(labels, np.int32, "labels"), int(n_chunks)), "hough_run_host_chunked")


def hough_measure_smem_atomic_peak(device: int = 0, millis: float = 20.0) -> Tuple[float, float]:
    """(conflict-free shared-memory atomic adds per second over the whole chip, SM clock in MHz seen meanwhile)."""
    ops, mhz = ctypes.c_double(0), ctypes.c_double(0)
    _check(load_library().hough_measure_smem_atomic_peak(device, millis, ctypes.byref(ops), ctypes.byref(mhz)),
           "hough_measure_smem_atomic_peak")
    return ops.value, mhz.value


def hough_version() -> int:
    return int(load_library().hough_version())


def candidates_to_numpy(cands: torch.Tensor) -> np.ndarray:
    """int32 [E, K, 8] device/host tensor -> numpy structured array [E, K] of CANDIDATE_DTYPE (a copy on the host)."""
    a = cands.detach().cpu().numpy()
    return np.ascontiguousarray(a).view(CANDIDATE_DTYPE).reshape(a.shape[0], a.shape[1])


def plan_for_workload(wl, n_events: int, n_hits: int, max_hits_per_event: int, device: int = 0, flags: int = 0) -> Plan:
    """Plan of a synth.Workload (grid, threshold, window, K of SURVEY.md Sec. 8(d))."""
    return hough_plan_create(wl.n_theta, wl.n_rho, wl.rho_min, wl.rho_max, wl.coord_max, wl.vote_threshold, wl.assign_window,
                             wl.max_candidates, max(1, n_events), max(0, n_hits), max_hits_per_event,
                             HOUGH_U16 if wl.count_dtype == "u16" else HOUGH_I32, wl.hit_frac_bits, -1, device, flags)


def hough_refit_tracks(plan: Plan, u: torch.Tensor, v: torch.Tensor, offsets: torch.Tensor, n_found: torch.Tensor,
                       labels: torch.Tensor, plane_origin: float, plane_pitch: float, n_planes: int, min_run: int = 5,
                       wrap: bool = False, fits: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """fits int32 [E, K, 8] -- the 32-byte hough_fit_t records as words (see fits_to_numpy); rows beyond min(n_found, K) untouched."""
    E = _n_events(offsets)
    if fits is None:
        fits = torch.zeros((E, plan.K, 8), dtype=torch.int32, device=plan.device)
    g = hough_plane_geometry_t(plane_origin, plane_pitch, n_planes, min_run, int(bool(wrap)), 0)
    _check(load_library().hough_refit_tracks(plan.handle, _dev(plan, u, torch.float32, "u"), _dev(plan, v, torch.float32, "v"),
                                             _dev(plan, offsets, torch.int64, "offsets"), E, _dev(plan, n_found, torch.int32, "n_found"),
                                             _dev(plan, labels, torch.int32, "labels"), ctypes.byref(g),
                                             _dev(plan, fits, torch.int32, "fits"), _stream_ptr(plan, stream)), "hough_refit_tracks")
    return fits


def fits_to_numpy(fits: torch.Tensor) -> np.ndarray:
    """int32 [E, K, 8] tensor -> numpy structured array [E, K] of FIT_DTYPE (a copy on the host)."""
    a = np.ascontiguousarray(fits.detach().cpu().numpy())
    return a.view(FIT_DTYPE).reshape(a.shape[0], a.shape[1])


class FrontEnd:
    """Owner of a hough_frontend_t* (time slicing + phi = atan2(y, x))."""

    def __init__(self, handle: int, desc: hough_frontend_desc_t):
        self.handle = ctypes.c_void_p(handle)
        self.desc = desc
        self.device = torch.device("cuda", desc.device)
        self.windows_per_fill = desc.windows_per_fill

    def __del__(self):
        try:
            hough_frontend_destroy(self)
        except Exception:
            pass


def hough_frontend_create(t0: float, window_width: float, window_step: float, windows_per_fill: int, max_fills: int,
                          max_hits: int, xy_max: float = 512.0, device: int = 0) -> FrontEnd:
    d = hough_frontend_desc_t(t0, window_width, window_step, windows_per_fill, xy_max, max_fills, max_hits, device, 0)
    h = ctypes.c_void_p()
    _check(load_library().hough_frontend_create(ctypes.byref(d), ctypes.byref(h)), "hough_frontend_create")
    return FrontEnd(h.value, d)


def hough_frontend_destroy(fe: FrontEnd) -> None:
    if fe.handle is not None and fe.handle.value:
        h, fe.handle = fe.handle, None
        _check(load_library().hough_frontend_destroy(h), "hough_frontend_destroy")


def hough_frontend_slice(fe: FrontEnd, x: torch.Tensor, y: torch.Tensor, z: torch.Tensor, t: torch.Tensor,
                         fill_offsets: torch.Tensor, capacity: Optional[int] = None, stream=None):
    """(u [capacity] fp32, v [capacity] fp32, src [capacity] int32, offsets [n_fills * windows_per_fill + 1] int64) on the device.
    Only the first offsets[-1] entries of u, v, src are meaningful; capacity defaults to ceil(width / step) * n_hits."""
    n_fills = _n_events(fill_offsets)
    n = x.numel()
    if capacity is None:
        capacity = n * int(-(-fe.desc.window_width // fe.desc.window_step))
    u = torch.empty(max(capacity, 1), dtype=torch.float32, device=fe.device)
    v = torch.empty(max(capacity, 1), dtype=torch.float32, device=fe.device)
    src = torch.empty(max(capacity, 1), dtype=torch.int32, device=fe.device)
    offsets = torch.empty(n_fills * fe.windows_per_fill + 1, dtype=torch.int64, device=fe.device)
    s = stream if stream is not None else torch.cuda.current_stream(fe.device)
    _check(load_library().hough_frontend_slice(fe.handle, _dev(fe, x, torch.float32, "x"), _dev(fe, y, torch.float32, "y"),
                                               _dev(fe, z, torch.float32, "z"), _dev(fe, t, torch.float32, "t"),
                                               _dev(fe, fill_offsets, torch.int64, "fill_offsets"), n_fills, n,
                                               ctypes.c_void_p(u.data_ptr()), ctypes.c_void_p(v.data_ptr()),
                                               ctypes.c_void_p(src.data_ptr()), ctypes.c_void_p(offsets.data_ptr()), capacity,
                                               ctypes.c_void_p(s.cuda_stream)), "hough_frontend_slice")
    return u, v, src, offsets


def hough_frontend_status(fe: FrontEnd, stream=None) -> int:
    out = ctypes.c_int32(0)
    s = stream if stream is not None else torch.cuda.current_stream(fe.device)
    _check(load_library().hough_frontend_status(fe.handle, ctypes.byref(out), ctypes.c_void_p(s.cuda_stream)), "hough_frontend_status")
    return out.value


def hough_find_tracks_peeloff(plan: Plan, u: torch.Tensor, v: torch.Tensor, offsets: torch.Tensor, stream=None):
    """The paper's one-track-at-a-time peak rule (variant).  -> (cands int32 [E, K, 8], n_found int32 [E], labels int32 [N])."""
    E = _n_events(offsets)
    cands = torch.zeros((E, plan.K, CANDIDATE_WORDS), dtype=torch.int32, device=plan.device)
    n_found = torch.zeros(E, dtype=torch.int32, device=plan.device)
    labels = torch.empty(max(u.numel(), 1), dtype=torch.int32, device=plan.device)
    _check(load_library().hough_find_tracks_peeloff(plan.handle, _dev(plan, u, torch.float32, "u"), _dev(plan, v, torch.float32, "v"),
                                                    _dev(plan, offsets, torch.int64, "offsets"), E,
                                                    _dev(plan, cands, torch.int32, "cands"), _dev(plan, n_found, torch.int32, "n_found"),
                                                    _dev(plan, labels, torch.int32, "labels"), _stream_ptr(plan, stream)),
           "hough_find_tracks_peeloff")
    return cands, n_found, labels[: u.numel()]


def hough_find_two_stage(plan: Plan, u: torch.Tensor, v: torch.Tensor, offsets: torch.Tensor, coarse_theta: int, coarse_rho: int,
                         stream=None):
    """The paper's coarse -> fine two-stage histogram (variant).  -> (cands int32 [E, K, 8], n_found int32 [E])."""
    E = _n_events(offsets)
    cands = torch.zeros((E, plan.K, CANDIDATE_WORDS), dtype=torch.int32, device=plan.device)
    n_found = torch.zeros(E, dtype=torch.int32, device=plan.device)
    _check(load_library().hough_find_two_stage(plan.handle, _dev(plan, u, torch.float32, "u"), _dev(plan, v, torch.float32, "v"),
                                               _dev(plan, offsets, torch.int64, "offsets"), E, coarse_theta, coarse_rho,
                                               _dev(plan, cands, torch.int32, "cands"), _dev(plan, n_found, torch.int32, "n_found"),
                                               _stream_ptr(plan, stream)), "hough_find_two_stage")
    return cands, n_found
