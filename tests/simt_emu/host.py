"""TEST INFRASTRUCTURE: the product's C ABI on the CPU.  libhough_hostemu.so = the product's HOST code
(paper_2607_04067_b200/csrc/hough_api.cu: handles, options, planner, launch set-up, hough_run_host's staging)
compiled by g++ against tests/simt_emu/fake_cuda_runtime.h, every kernel launch executed by the SIMT emulator on the
kernel source (host_emu.cpp).  The tests call the same entry points as a GPU user would, numpy arrays standing in for
device buffers, and compare with the oracle: what emu_main.cpp checks for the kernel alone, this checks for the host
code in front of it.  `race=True` loads the race-check build (simt_shim.h): every launch is also a racecheck + initcheck.
Not a product path: the package never builds or loads this library."""
import ctypes
import os
import subprocess
import threading

import numpy as np

from . import FLAGS, HERE, ROOT, SOURCES

HOST_SOURCES = [os.path.join(HERE, "host_emu.cpp"), os.path.join(HERE, "fake_cuda_runtime.h"), os.path.join(HERE, "simt_shim.h"),
                os.path.join(ROOT, "paper_2607_04067_b200", "csrc", "hough_api.cu"), SOURCES[2], SOURCES[3],
                os.path.join(ROOT, "include", "hough_debug.h"), os.path.abspath(__file__)]
_LOCK = threading.Lock()
_libs = {}


def build(race: bool = False, force: bool = False) -> str:
    with _LOCK:
        return _build_unlocked(race, force)


def _build_unlocked(race: bool = False, force: bool = False) -> str:
    lib = os.path.join(HERE, "libhough_hostemu_race.so" if race else "libhough_hostemu.so")
    if True:
        if not force and os.path.exists(lib) and all(os.path.getmtime(s) <= os.path.getmtime(lib) for s in HOST_SOURCES):
            return lib
        tmp = lib + ".tmp.%d" % os.getpid()
        # race: the compiler's -fsanitize=thread instrumentation only; the link line must not add ThreadSanitizer's runtime
        obj = tmp + ".o"
        subprocess.check_call(["g++", *FLAGS, "-fPIC", "-Wno-subobject-linkage", *(["-fsanitize=thread"] if race else []), "-x", "c++", "-c", "-o", obj, HOST_SOURCES[0]])
        subprocess.check_call(["g++", "-shared", "-o", tmp, obj])
        os.remove(obj)
        os.replace(tmp, lib)
        return lib


def load(race: bool = False):
    """The library with the product binding's own argument declarations."""
    import paper_2607_04067_b200 as hb
    if race not in _libs:
        lib = hb._declare_abi(ctypes.CDLL(build(race)))
        lib.hough_hostemu_counters.restype = None
        lib.hough_hostemu_counters.argtypes = [ctypes.POINTER(ctypes.c_longlong)]
        vp, cll = ctypes.c_void_p, ctypes.c_longlong
        lib.hough_hostemu_malloc.restype = vp
        lib.hough_hostemu_malloc.argtypes = [cll]
        lib.hough_hostemu_free.restype = None
        lib.hough_hostemu_free.argtypes = [vp]
        for f in (lib.hough_hostemu_upload, lib.hough_hostemu_poke, lib.hough_hostemu_download):
            f.restype = None
            f.argtypes = [vp, vp, cll]
        _libs[race] = lib
    return _libs[race]


def counters(lib):
    out = (ctypes.c_longlong * 4)()
    lib.hough_hostemu_counters(out)
    return {"malloc": out[0], "free": out[1], "launches": out[2], "reports": out[3]}


def _p(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


class DeviceBuffers:
    """The caller's device buffers of one call: emulated device allocations (guard page behind the end) holding copies
    of numpy arrays.  Inputs are uploaded; outputs are poked (their poison does not count as written for the initcheck)
    and downloaded afterwards."""

    def __init__(self, lib):
        self.lib, self.items = lib, []

    def put(self, a, output=False):
        if a is None:
            return None
        p = self.lib.hough_hostemu_malloc(a.nbytes)
        if not p:
            raise MemoryError("hough_hostemu_malloc")
        (self.lib.hough_hostemu_poke if output else self.lib.hough_hostemu_upload)(p, a.ctypes.data, a.nbytes)
        self.items.append((p, a, output))
        return ctypes.c_void_p(p)

    def finish(self):
        for p, a, output in self.items:
            if output:
                self.lib.hough_hostemu_download(a.ctypes.data, p, a.nbytes)
            self.lib.hough_hostemu_free(p)
        self.items = []


class Handle:
    """hough_create ... hough_destroy through the emulated ABI; numpy in, numpy out."""

    def __init__(self, n_theta, n_rho, rho_max, threshold, window, table, max_peaks=64, acc_dtype="u16", conformal_scale=1,
                 cluster_size=0, ctas_per_sm=0, vote_path=0, peak_mode=0, rel_permille=None, nms_radius=None, theta_wrap=False,
                 keep_mode=0, keep_tol=None, b_field=None, staging=0, scheduler=0, select_mode=0, race=False):
        import paper_2607_04067_b200 as hb
        self.hb, self.lib = hb, load(race)
        self.n_theta, self.n_rho, self.max_peaks = n_theta, n_rho, max_peaks
        self.ctx = self.lib.hough_create(n_theta, n_rho, float(np.float32(rho_max)), threshold, window)
        if not self.ctx:
            raise RuntimeError("hough_create failed: %s" % self.lib.hough_last_error().decode())
        acc = {"auto": hb.HOUGH_ACC_AUTO, "u16": hb.HOUGH_ACC_U16, "u32": hb.HOUGH_ACC_U32}[acc_dtype]
        for key, v in ((hb.HOUGH_OPT_MAX_PEAKS, max_peaks), (hb.HOUGH_OPT_ACC_DTYPE, acc), (hb.HOUGH_OPT_CONFORMAL_SCALE, conformal_scale),
                       (hb.HOUGH_OPT_CLUSTER_SIZE, cluster_size), (hb.HOUGH_OPT_CTAS_PER_SM, ctas_per_sm), (hb.HOUGH_OPT_VOTE_PATH, vote_path),
                       (hb.HOUGH_OPT_PEAK_MODE, peak_mode), (hb.HOUGH_OPT_REL_THRESHOLD_PERMILLE, rel_permille), (hb.HOUGH_OPT_NMS_RADIUS, nms_radius),
                       (hb.HOUGH_OPT_THETA_WRAP, int(bool(theta_wrap))), (hb.HOUGH_OPT_KEEP_MODE, keep_mode), (hb.HOUGH_OPT_STAGING, staging),
                       (hb.HOUGH_OPT_SCHEDULER, scheduler), (hb.HOUGH_OPT_SELECT_MODE, select_mode)):
            if v is not None and v != 0 or key in (hb.HOUGH_OPT_MAX_PEAKS, hb.HOUGH_OPT_ACC_DTYPE):
                self.check(self.lib.hough_set_option(self.ctx, key, int(v)), "hough_set_option(%d)" % key)
        for key, v in ((hb.HOUGH_OPTF_KEEP_TOL, keep_tol), (hb.HOUGH_OPTF_B_FIELD_TESLA, b_field)):
            if v is not None:
                self.check(self.lib.hough_set_option_f64(self.ctx, key, float(v)), "hough_set_option_f64(%d)" % key)
        c, s = (np.ascontiguousarray(t, dtype=np.float32) for t in table)
        self.check(self.lib.hough_set_trig_table(self.ctx, _p(c), _p(s)), "hough_set_trig_table")

    def check(self, rc, what):
        if rc != self.hb.HOUGH_OK:
            raise self.hb.HoughError("%s failed: %s (%s)" % (what, self.lib.hough_strerror(rc).decode(), self.lib.hough_last_error().decode()))

    def info(self, key):
        return int(self.lib.hough_get_info(self.ctx, key))

    def outputs(self, n_total, n_events, accum=False):
        """Poisoned output arrays, as tests/test_parity_gpu.py::gpu_run prepares them."""
        o = {"keep": np.full(n_total, 7, np.uint8), "peaks": np.full((n_events, self.max_peaks, 2), -1, np.int32),
             "counts": np.full((n_events, 2), -99, np.int32), "kept_xy": np.zeros((n_total, 2), np.float32),
             "kept_idx": np.full(n_total, -5, np.int32)}
        if accum:
            o["accum"] = np.zeros((n_events, self.n_theta, self.n_rho), np.int32)
        return o

    def run(self, xy, off, out=None, accum=False, kept=True, n_events=None):
        hb = self.hb
        xy = np.ascontiguousarray(xy, dtype=np.float32).reshape(-1, 2)
        off = np.ascontiguousarray(off, dtype=np.int32)
        n_events = len(off) - 1 if n_events is None else n_events
        out = out or self.outputs(len(xy), n_events, accum)
        dev = DeviceBuffers(self.lib)
        try:
            io = hb.hough_io(dev.put(xy), dev.put(off), n_events, dev.put(out["keep"], True), dev.put(out["peaks"], True),
                             dev.put(out["counts"], True), dev.put(out["kept_xy"], True) if kept else None,
                             dev.put(out["kept_idx"], True) if kept else None, dev.put(out.get("accum"), True))
            self.check(self.lib.hough_run_ex(self.ctx, ctypes.byref(io), None), "hough_run_ex")
        finally:
            dev.finish()
        return out

    def circles(self, xy, off, out):
        xy = np.ascontiguousarray(xy, dtype=np.float32).reshape(-1, 2)
        off = np.ascontiguousarray(off, dtype=np.int32)
        n_events = len(off) - 1
        circ = np.zeros((n_events, self.max_peaks), self.hb.circle_dtype())
        dev = DeviceBuffers(self.lib)
        try:
            self.check(self.lib.hough_circles(self.ctx, dev.put(xy), dev.put(off), n_events, dev.put(out["peaks"]), dev.put(out["counts"]),
                                              dev.put(circ, True), None), "hough_circles")
        finally:
            dev.finish()
        return circ

    def run_host(self, xy, off, n_events, keep, peaks, counts, kept_xy=None, kept_idx=None, stream=0):
        """off may be a VIEW into a longer offsets array (absolute offsets into xy), as hough_run_host allows."""
        self.check(self.lib.hough_run_host(self.ctx, _p(xy), ctypes.c_void_p(off.ctypes.data), n_events, _p(keep),
                                           ctypes.c_void_p(peaks.ctypes.data), ctypes.c_void_p(counts.ctypes.data), _p(kept_xy), _p(kept_idx),
                                           ctypes.c_void_p(stream)), "hough_run_host")

    def close(self):
        if self.ctx:
            self.lib.hough_destroy(self.ctx)
            self.ctx = None
