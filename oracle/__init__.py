"""Python face of the CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It never imports
paper_2607_04067_b200 and shares no code with it.  See hough_oracle.cpp for
the steps S1..S6 and the passages of PAPER.md they restate.
"""
import ctypes
from dataclasses import dataclass

import numpy as np

from .build import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build())
        f32p = ctypes.POINTER(ctypes.c_float)
        lib.oracle_run.restype = ctypes.c_int
        lib.oracle_run.argtypes = [
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
            ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_int, ctypes.c_int,
            ctypes.c_int, ctypes.c_int, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
        lib.oracle_conformal.restype = None
        lib.oracle_conformal.argtypes = [ctypes.c_float, ctypes.c_float, ctypes.c_int, f32p, f32p]
        lib.oracle_rho_bin.restype = ctypes.c_int
        lib.oracle_rho_bin.argtypes = [ctypes.c_float] * 5 + [ctypes.c_int]
        vp, ci = ctypes.c_void_p, ctypes.c_int
        lib.oracle_find_peaks.restype = ci
        lib.oracle_find_peaks.argtypes = [vp, ci, ci, ci, ci, vp]
        lib.oracle_find_peaks_ex.restype = ci
        lib.oracle_find_peaks_ex.argtypes = [vp, ci, ci, ci, ci, vp, vp]
        lib.oracle_run_ex.restype = ci
        lib.oracle_run_ex.argtypes = [vp, vp, ci, ci, ci, ctypes.c_float, ci, ci, ci, ci, ci, vp, vp, vp,
                                      ctypes.c_double, ctypes.c_double, vp, vp, vp, vp, vp, vp, vp, ci]
        _lib = lib
    return _lib


@dataclass
class OracleResult:
    keep: np.ndarray       # [n_total] u8
    peaks: np.ndarray      # [n_events, max_peaks, 3] u32 (theta_bin, rho_bin, votes); rows >= stored are 0
    counts: np.ndarray     # [n_events, 2] i32 {n_peaks untruncated, n_kept}
    kept_xy: np.ndarray    # [n_total, 2] f32; event e's kept hits start at offsets[e]
    kept_idx: np.ndarray   # [n_total] i32; index within the event
    accum: np.ndarray      # [n_events, n_theta, n_rho] u32 or None


def run(xy, offsets, n_theta, n_rho, rho_max, threshold, window, cos_t, sin_t,
        max_peaks=64, conformal_scale=1, acc_u16=True, want_accum=False, n_threads=1):
    """Runs S1..S6 on a batch of events.  All arrays are numpy; rho_max is
    rounded to fp32 here exactly as a C float argument would be."""
    lib = _load()
    xy = np.ascontiguousarray(xy, dtype=np.float32).reshape(-1, 2)
    offsets = np.ascontiguousarray(offsets, dtype=np.int32)
    cos_t = np.ascontiguousarray(cos_t, dtype=np.float32)
    sin_t = np.ascontiguousarray(sin_t, dtype=np.float32)
    assert cos_t.shape == (n_theta,) and sin_t.shape == (n_theta,)
    n_events = offsets.shape[0] - 1
    n_total = int(offsets[-1]) if n_events >= 0 and offsets.size else 0
    assert xy.shape[0] >= n_total
    keep = np.zeros(n_total, dtype=np.uint8)
    peaks = np.zeros((max(n_events, 0), max_peaks, 3), dtype=np.uint32)
    counts = np.zeros((max(n_events, 0), 2), dtype=np.int32)
    kept_xy = np.zeros((n_total, 2), dtype=np.float32)
    kept_idx = np.zeros(n_total, dtype=np.int32)
    accum = np.zeros((max(n_events, 0), n_theta, n_rho), dtype=np.uint32) if want_accum else None
    rc = lib.oracle_run(
        xy.ctypes.data, offsets.ctypes.data, n_events,
        n_theta, n_rho, ctypes.c_float(np.float32(rho_max)), threshold, window,
        max_peaks, conformal_scale, 1 if acc_u16 else 0,
        cos_t.ctypes.data, sin_t.ctypes.data,
        keep.ctypes.data, peaks.ctypes.data, counts.ctypes.data,
        kept_xy.ctypes.data, kept_idx.ctypes.data,
        accum.ctypes.data if accum is not None else None, n_threads)
    if rc != 0:
        raise ValueError("oracle_run: bad argument")
    return OracleResult(keep, peaks, counts, kept_xy, kept_idx, accum)


def conformal(x, y, conformal_scale=1):
    lib = _load()
    u = ctypes.c_float()
    v = ctypes.c_float()
    lib.oracle_conformal(ctypes.c_float(np.float32(x)), ctypes.c_float(np.float32(y)), conformal_scale,
                         ctypes.byref(u), ctypes.byref(v))
    return np.float32(u.value), np.float32(v.value)


def rho_bin(u, v, c, s, rho_max, n_rho):
    lib = _load()
    f = lambda a: ctypes.c_float(np.float32(a))
    return lib.oracle_rho_bin(f(u), f(v), f(c), f(s), f(rho_max), n_rho)


# ---------------------------------------------------------------- the NEXT rows (hough_oracle_next.cpp)
CIRCLE_DTYPE = np.dtype([("x_c", "<f8"), ("y_c", "<f8"), ("r_c", "<f8"), ("pt", "<f8"), ("phi0", "<f8"),
                         ("charge", "<i4"), ("n_hits", "<i4")])     # 48 bytes, the layout of hough_circle


def _opts(peak_mode, rel_permille, nms_radius, theta_wrap, keep_mode):
    return np.array([peak_mode, rel_permille, nms_radius, int(bool(theta_wrap)), keep_mode], dtype=np.int32)


def run_ex(xy, offsets, n_theta, n_rho, rho_max, threshold, window, cos_t, sin_t, max_peaks=64, conformal_scale=1,
           acc_u16=True, want_accum=False, n_threads=1, peak_mode=0, rel_permille=500, nms_radius=1, theta_wrap=False,
           keep_mode=0, keep_tol=0.0, b_field=1.0, want_circles=False):
    """oracle.run plus the NEXT options (N1 circles, N2 relative threshold + iterative NMS, N4a theta wrap, N4b distance
    filter).  Returns (OracleResult, circles) with circles a [n_events, max_peaks] structured array or None."""
    lib = _load()
    xy = np.ascontiguousarray(xy, dtype=np.float32).reshape(-1, 2)
    offsets = np.ascontiguousarray(offsets, dtype=np.int32)
    cos_t = np.ascontiguousarray(cos_t, dtype=np.float32)
    sin_t = np.ascontiguousarray(sin_t, dtype=np.float32)
    n_events = offsets.shape[0] - 1
    n_total = int(offsets[-1])
    keep = np.zeros(n_total, dtype=np.uint8)
    peaks = np.zeros((n_events, max_peaks, 3), dtype=np.uint32)
    counts = np.zeros((n_events, 2), dtype=np.int32)
    kept_xy = np.zeros((n_total, 2), dtype=np.float32)
    kept_idx = np.zeros(n_total, dtype=np.int32)
    accum = np.zeros((n_events, n_theta, n_rho), dtype=np.uint32) if want_accum else None
    circ = np.zeros((n_events, max_peaks), dtype=CIRCLE_DTYPE) if want_circles else None
    opts = _opts(peak_mode, rel_permille, nms_radius, theta_wrap, keep_mode)
    rc = lib.oracle_run_ex(xy.ctypes.data, offsets.ctypes.data, n_events, n_theta, n_rho, ctypes.c_float(np.float32(rho_max)),
                           threshold, window, max_peaks, conformal_scale, 1 if acc_u16 else 0, cos_t.ctypes.data, sin_t.ctypes.data,
                           opts.ctypes.data, float(keep_tol), float(b_field), keep.ctypes.data, peaks.ctypes.data, counts.ctypes.data,
                           kept_xy.ctypes.data, kept_idx.ctypes.data, accum.ctypes.data if accum is not None else None,
                           circ.ctypes.data if circ is not None else None, n_threads)
    if rc != 0:
        raise ValueError("oracle_run_ex: bad argument")
    return OracleResult(keep, peaks, counts, kept_xy, kept_idx, accum), circ


def find_peaks(A, threshold, max_peaks=4096):
    """S3/S4 of hough_oracle.cpp on a caller-made accumulator [n_theta, n_rho].  Returns (n_peaks, peaks [min(n, max), 3])."""
    lib = _load()
    A = np.ascontiguousarray(A, dtype=np.uint32)
    out = np.zeros((max_peaks, 3), dtype=np.uint32)
    n = lib.oracle_find_peaks(A.ctypes.data, A.shape[0], A.shape[1], threshold, max_peaks, out.ctypes.data)
    return n, out[:min(n, max_peaks)]


def find_peaks_ex(A, threshold, max_peaks=4096, peak_mode=0, rel_permille=500, nms_radius=1, theta_wrap=False):
    """Peak finding of hough_oracle_next.cpp (3x3 with optional wrap, or relative threshold + iterative NMS)."""
    lib = _load()
    A = np.ascontiguousarray(A, dtype=np.uint32)
    out = np.zeros((max_peaks, 3), dtype=np.uint32)
    opts = _opts(peak_mode, rel_permille, nms_radius, theta_wrap, 0)
    n = lib.oracle_find_peaks_ex(A.ctypes.data, A.shape[0], A.shape[1], threshold, max_peaks, opts.ctypes.data, out.ctypes.data)
    return n, out[:min(n, max_peaks)]
