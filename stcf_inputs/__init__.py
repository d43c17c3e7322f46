"""Seeded synthetic inputs shared by the oracle and the CUDA path.

Holds no arithmetic of the method (no conformal map, no rho bins): only the
event generator (gen.cpp, recipe in DESIGN.md "Input recipe"), the five
workload configurations of BASELINE.json `configs`, and the host-built
cos/sin table that both sides receive as DATA (reading Q3).
"""
import ctypes
import os
import subprocess
from dataclasses import dataclass, replace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.cpp")
_LIB = os.path.join(_HERE, "libstcfgen.so")
_lib = None


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.stcf_generate.restype = ctypes.c_longlong
        lib.stcf_generate.argtypes = [
            ctypes.c_ulonglong, ctypes.c_longlong, ctypes.c_int,
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p]
        _lib = lib
    return _lib


# rho_max = 1/(2 * 0.167 m) in mm^-1: fp32 nearest to 1/334 (reading Q2).
RHO_MAX = np.float32(1.0) / np.float32(334.0)


@dataclass(frozen=True)
class Workload:
    """One entry of BASELINE.json `configs`: the event mix plus the Hough grid."""
    name: str
    n_events: int
    seed: int
    tracks: tuple          # (lo, hi) signal tracks per event, uniform
    pt_gev: tuple          # (lo, hi) log-uniform
    turns: tuple           # (lo, hi) repeats of a track's hit set
    bkg_lambda: float      # Poisson mean of background hits per event
    n_theta: int
    n_rho: int
    threshold: int
    window: int
    max_peaks: int
    acc_dtype: str         # "u16" | "u32"
    rho_max: float = float(RHO_MAX)
    sigma_mm: float = 0.13


CONFIGS = {
    0: Workload("cfg0_pr1_ref", 16, 1, (2, 2), (0.3, 1.5), (1, 1), 100.0, 180, 128, 20, 1, 64, "u16"),
    1: Workload("cfg1_nominal", 1000, 2, (1, 6), (0.1, 2.0), (1, 1), 600.0, 180, 256, 16, 1, 64, "u16"),
    2: Workload("cfg2_lowpt_curlers", 1000, 3, (2, 4), (0.05, 0.15), (1, 3), 600.0, 360, 256, 10, 1, 4096, "u16"),
    3: Workload("cfg3_high_occupancy", 1000, 4, (4, 10), (0.1, 2.0), (1, 1), 2500.0, 180, 256, 20, 2, 2048, "u32"),
    4: Workload("cfg4_sweep_180x256", 100000, 5, (1, 6), (0.1, 2.0), (1, 1), 600.0, 180, 256, 16, 1, 64, "u16"),
    5: Workload("cfg4_sweep_360x512", 100000, 5, (1, 6), (0.1, 2.0), (1, 1), 600.0, 360, 512, 16, 1, 64, "u16"),
}


def config(i: int, n_events: int = None) -> Workload:
    w = CONFIGS[i]
    return w if n_events is None else replace(w, n_events=n_events)


def generate(w: Workload, n_events: int = None, first_event: int = 0):
    """Returns (xy [N,2] f32, offsets [n+1] i32, truth [N] u8) for events
    [first_event, first_event+n_events) of workload `w` (seed = w.seed)."""
    lib = _load()
    n = w.n_events if n_events is None else n_events
    offsets = np.zeros(n + 1, dtype=np.int32)
    per_ev = w.tracks[1] * 48 * w.turns[1] + w.bkg_lambda + 12.0 * np.sqrt(w.bkg_lambda + 1.0) + 64
    cap = int(n * per_ev) + 1024
    while True:
        xy = np.empty((cap, 2), dtype=np.float32)
        truth = np.empty(cap, dtype=np.uint8)
        total = lib.stcf_generate(
            w.seed, first_event, n, w.tracks[0], w.tracks[1], w.pt_gev[0], w.pt_gev[1],
            w.turns[0], w.turns[1], w.bkg_lambda, w.sigma_mm,
            xy.ctypes.data, truth.ctypes.data, cap, offsets.ctypes.data)
        if total <= cap:
            return xy[:total].copy(), offsets, truth[:total].copy()
        cap = int(total)


def trig_table(n_theta: int):
    """theta_j = j*pi/n_theta (left edges of equal bins on [0, pi), PAPER.md:73,
    :92; reading Q3), evaluated in double and rounded once to fp32.  Built once
    by the harness and handed to BOTH the oracle and hough_set_trig_table."""
    theta = np.arange(n_theta, dtype=np.float64) * (np.pi / n_theta)
    return np.cos(theta).astype(np.float32), np.sin(theta).astype(np.float32)
