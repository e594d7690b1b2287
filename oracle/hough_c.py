"""ctypes front end of oracle/hough_oracle.c (the plain C oracle) and its gcc build step.

TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT (see hough_oracle.c).  Nothing under
paper_2511_02742_b200/ imports this module.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

from .hough_def import Params

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hough_oracle.c")
_LIB = os.path.join(_HERE, "libhough_oracle.so")

CAND_DTYPE = np.dtype([("theta_bin", "<i4"), ("rho_bin", "<i4"), ("votes", "<i4"), ("cluster_root", "<i4"),
                       ("cluster_nbins", "<i4"), ("theta", "<f4"), ("rho", "<f4"), ("reserved", "<i4")])
assert CAND_DTYPE.itemsize == 32


class _CParams(ctypes.Structure):
    _fields_ = [("n_theta", ctypes.c_int32), ("n_rho", ctypes.c_int32),
                ("rho_min", ctypes.c_double), ("rho_max", ctypes.c_double), ("coord_max", ctypes.c_double),
                ("vote_threshold", ctypes.c_int32), ("assign_window", ctypes.c_double),
                ("max_candidates", ctypes.c_int32), ("hit_frac_bits", ctypes.c_int32), ("acc_frac_bits", ctypes.c_int32),
                ("theta_min", ctypes.c_double), ("theta_max", ctypes.c_double),
                ("theta_wrap", ctypes.c_int32), ("reserved", ctypes.c_int32)]


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (plain -O2, no fast-math, no FMA contraction, single-threaded)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fno-fast-math", "-ffp-contract=off",
                               "-Wall", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        P = ctypes.POINTER(_CParams)
        vp = ctypes.c_void_p
        L.ho_default_frac_bits.argtypes = [P]
        L.ho_default_frac_bits.restype = ctypes.c_int
        L.ho_constants.argtypes = [P, vp, vp, vp]
        L.ho_constants.restype = ctypes.c_int
        L.ho_vote_event.argtypes = [P, vp, vp, ctypes.c_int64, vp]
        L.ho_vote_event.restype = ctypes.c_int
        L.ho_find_clusters_event.argtypes = [P, vp, vp, vp]
        L.ho_find_clusters_event.restype = ctypes.c_int
        L.ho_assign_event.argtypes = [P, vp, vp, ctypes.c_int64, vp, ctypes.c_int32, vp]
        L.ho_assign_event.restype = ctypes.c_int
        L.ho_digest.argtypes = [vp, ctypes.c_int32, ctypes.c_int32]
        L.ho_digest.restype = ctypes.c_uint64
        L.ho_run_batch.argtypes = [P, vp, vp, vp, ctypes.c_int64, vp, vp, vp, vp, vp]
        L.ho_run_batch.restype = ctypes.c_int
        _lib = L
    return _lib


def _cp(p: Params) -> _CParams:
    return _CParams(p.n_theta, p.n_rho, p.rho_min, p.rho_max, p.coord_max, p.vote_threshold, p.assign_window,
                    p.max_candidates, p.hit_frac_bits, p.acc_frac_bits, p.theta_min, p.theta_max, int(p.theta_wrap), 0)


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _check(rc: int):
    if rc != 0:
        raise RuntimeError({-1: "int32 bound of the fixed-point design violated", -2: "out of memory",
                            -3: "bad arguments"}.get(rc, f"oracle error {rc}"))


def constants(p: Params):
    """(H, F, O_q, W_q, C_q[int64], S_q[int64])."""
    Cq = np.zeros(p.n_theta, np.int64)
    Sq = np.zeros(p.n_theta, np.int64)
    scal = np.zeros(4, np.int64)
    cp = _cp(p)
    _check(lib().ho_constants(ctypes.byref(cp), _ptr(Cq), _ptr(Sq), _ptr(scal)))
    return int(scal[0]), int(scal[1]), int(scal[2]), int(scal[3]), Cq, Sq


def vote_event(u: np.ndarray, v: np.ndarray, p: Params) -> np.ndarray:
    u = np.ascontiguousarray(u, np.float32)
    v = np.ascontiguousarray(v, np.float32)
    acc = np.zeros((p.n_theta, p.n_rho), np.int32)
    cp = _cp(p)
    _check(lib().ho_vote_event(ctypes.byref(cp), _ptr(u), _ptr(v), len(u), _ptr(acc)))
    return acc


def find_clusters_event(acc: np.ndarray, p: Params):
    acc = np.ascontiguousarray(acc, np.int32)
    cands = np.zeros(p.max_candidates, CAND_DTYPE)
    nf = np.zeros(1, np.int32)
    cp = _cp(p)
    _check(lib().ho_find_clusters_event(ctypes.byref(cp), _ptr(acc), _ptr(cands), _ptr(nf)))
    return cands[: min(int(nf[0]), p.max_candidates)], int(nf[0])


def assign_event(u: np.ndarray, v: np.ndarray, cands: np.ndarray, p: Params) -> np.ndarray:
    u = np.ascontiguousarray(u, np.float32)
    v = np.ascontiguousarray(v, np.float32)
    cands = np.ascontiguousarray(cands, CAND_DTYPE)
    labels = np.zeros(len(u), np.int32)
    cp = _cp(p)
    _check(lib().ho_assign_event(ctypes.byref(cp), _ptr(u), _ptr(v), len(u), _ptr(cands), len(cands), _ptr(labels)))
    return labels


def digest(acc: np.ndarray) -> int:
    acc = np.ascontiguousarray(acc, np.int32)
    return int(lib().ho_digest(_ptr(acc), acc.shape[0], acc.shape[1]))


def run_batch(u: np.ndarray, v: np.ndarray, offsets: np.ndarray, p: Params, want_cands: bool = True,
              want_labels: bool = True, want_digest: bool = False, want_acc: bool = False):
    """Whole path over a batch.  Returns dict(cands [E][K], n_found [E], labels [N], digest [E], acc [E][n_theta][n_rho])."""
    u = np.ascontiguousarray(u, np.float32)
    v = np.ascontiguousarray(v, np.float32)
    offsets = np.ascontiguousarray(offsets, np.int64)
    E = len(offsets) - 1
    out = {}
    cands = np.zeros((E, p.max_candidates), CAND_DTYPE) if want_cands else None
    n_found = np.zeros(E, np.int32) if (want_cands or want_labels) else None
    labels = np.zeros(len(u), np.int32) if want_labels else None
    dig = np.zeros(E, np.uint64) if want_digest else None
    acc = np.zeros((E, p.n_theta, p.n_rho), np.int32) if want_acc else None
    cp = _cp(p)
    _check(lib().ho_run_batch(ctypes.byref(cp), _ptr(u), _ptr(v), _ptr(offsets), E, _ptr(cands), _ptr(n_found),
                              _ptr(labels), _ptr(dig), _ptr(acc)))
    out.update(cands=cands, n_found=n_found, labels=labels, digest=dig, acc=acc)
    return out
