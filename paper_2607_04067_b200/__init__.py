"""paper_2607_04067_b200 -- thin Python binding of the C ABI in include/hough.h.

Argument marshalling only: every step of the hot path (conformal map, rho
matrix, voting, peaks, hit selection, compaction) runs in the CUDA kernels of
libhough_b200.so.  PyTorch is used for device memory and streams.  There is no
CPU fallback: if the library cannot be built/loaded or no CUDA device is
present, calls raise.  This package never imports oracle/.
"""
import ctypes
import os

from . import build as _build

HOUGH_OK = 0
HOUGH_ERR_INVALID_ARG = -1
HOUGH_ERR_UNSUPPORTED = -2
HOUGH_ERR_CUDA = -3
HOUGH_ERR_NOMEM = -4

HOUGH_OPT_MAX_PEAKS = 1
HOUGH_OPT_ACC_DTYPE = 2
HOUGH_OPT_CONFORMAL_SCALE = 3
HOUGH_OPT_CLUSTER_SIZE = 4
HOUGH_OPT_CTAS_PER_SM = 5
HOUGH_OPT_VOTE_PATH = 6
HOUGH_OPT_PEAK_MODE = 7
HOUGH_OPT_REL_THRESHOLD_PERMILLE = 8
HOUGH_OPT_NMS_RADIUS = 9
HOUGH_OPT_THETA_WRAP = 10
HOUGH_OPT_KEEP_MODE = 11
HOUGH_OPT_STAGING = 12
HOUGH_OPT_SCHEDULER = 13
HOUGH_OPT_SELECT_MODE = 14
HOUGH_OPTF_KEEP_TOL = 1
HOUGH_OPTF_B_FIELD_TESLA = 2
HOUGH_ACC_AUTO, HOUGH_ACC_U16, HOUGH_ACC_U32 = 0, 1, 2

HOUGH_INFO_CLUSTER_SIZE = 1
HOUGH_INFO_THREADS = 2
HOUGH_INFO_SMEM_BYTES = 3
HOUGH_INFO_CTAS_PER_SM = 4
HOUGH_INFO_GRID_MAX = 5
HOUGH_INFO_ACC_BITS = 6
HOUGH_INFO_MAX_PEAKS = 7
HOUGH_INFO_CHUNK_HITS = 8
HOUGH_INFO_SM_COUNT = 9
HOUGH_INFO_LAUNCHES = 10

# what each header under include/ declares, and which library exports it
EXPORTS = [            # include/hough.h -> libhough_b200.so (the product ABI)
    "hough_create", "hough_set_option", "hough_set_option_f64", "hough_set_trig_table", "hough_get_info", "hough_run", "hough_run_ex",
    "hough_circles", "hough_run_host", "hough_destroy", "hough_strerror", "hough_last_error", "hough_version",
]
DEBUG_EXPORTS = ["hough_plan_describe", "hough_debug_tame_bounds", "hough_debug_bounds_enabled"]   # include/hough_debug.h, same library
BENCH_EXPORTS = ["hough_bench_shared_atomics", "hough_bench_vote_loop", "hough_bench_issue_rate"]   # include/hough_bench.h -> libhough_bench.so


class hough_io(ctypes.Structure):
    _fields_ = [
        ("d_xy", ctypes.c_void_p), ("d_event_offsets", ctypes.c_void_p), ("n_events", ctypes.c_int32),
        ("d_keep_mask", ctypes.c_void_p), ("d_peaks", ctypes.c_void_p), ("d_counts", ctypes.c_void_p),
        ("d_kept_xy", ctypes.c_void_p), ("d_kept_idx", ctypes.c_void_p), ("d_accum_dump", ctypes.c_void_p),
    ]


class HoughError(RuntimeError):
    pass


_lib = None
_bench_lib = None


def flavor() -> str:
    """Which build of the product library this process uses: "release" (default), "dbg" (every shared-memory
    offset checked, HOUGH_B200_FLAVOR=dbg) or "diag" (bench-only phase-skipping diagnostics)."""
    f = os.environ.get("HOUGH_B200_FLAVOR", "release")
    if f not in ("release", "dbg", "diag"):
        raise HoughError("HOUGH_B200_FLAVOR must be release, dbg or diag (got %r)" % f)
    return f


def lib_path() -> str:
    return _build.lib_path(flavor())


def load_library():
    """Loads (building first if the sources are newer) libhough_b200.so.  Raises if that fails."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build(flavor())
    _lib = _declare_abi(ctypes.CDLL(path))
    return _lib


def _declare_abi(lib):
    """Argument and result types of every entry point of include/hough.h and include/hough_debug.h."""
    vp, ci, cll = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong
    lib.hough_create.restype = vp
    lib.hough_create.argtypes = [ci, ci, ctypes.c_float, ci, ci]
    lib.hough_set_option.restype = ci
    lib.hough_set_option.argtypes = [vp, ci, cll]
    lib.hough_set_option_f64.restype = ci
    lib.hough_set_option_f64.argtypes = [vp, ci, ctypes.c_double]
    lib.hough_circles.restype = ci
    lib.hough_circles.argtypes = [vp, vp, vp, ci, vp, vp, vp, vp]
    lib.hough_set_trig_table.restype = ci
    lib.hough_set_trig_table.argtypes = [vp, vp, vp]
    lib.hough_get_info.restype = cll
    lib.hough_get_info.argtypes = [vp, ci]
    lib.hough_run.restype = ci
    lib.hough_run.argtypes = [vp, vp, vp, ci, vp, vp, vp, vp]
    lib.hough_run_ex.restype = ci
    lib.hough_run_ex.argtypes = [vp, ctypes.POINTER(hough_io), vp]
    lib.hough_run_host.restype = ci
    lib.hough_run_host.argtypes = [vp, vp, vp, ci, vp, vp, vp, vp, vp, vp]
    lib.hough_destroy.restype = None
    lib.hough_destroy.argtypes = [vp]
    lib.hough_strerror.restype = ctypes.c_char_p
    lib.hough_strerror.argtypes = [ci]
    lib.hough_last_error.restype = ctypes.c_char_p
    lib.hough_last_error.argtypes = []
    lib.hough_version.restype = ctypes.c_char_p
    lib.hough_version.argtypes = []
    lib.hough_plan_describe.restype = ci
    lib.hough_plan_describe.argtypes = [ci, ci, ci, ci, ci, ci, ctypes.POINTER(cll), ci]
    lib.hough_debug_tame_bounds.restype = ci
    lib.hough_debug_tame_bounds.argtypes = [ci, ctypes.c_float, ctypes.c_float, ctypes.c_float, ctypes.POINTER(ctypes.c_float)]
    lib.hough_debug_bounds_enabled.restype = ci
    lib.hough_debug_bounds_enabled.argtypes = []
    return lib


def load_bench_library():
    """Loads libhough_bench.so (measurement aids, include/hough_bench.h); not needed by the product path."""
    global _bench_lib
    if _bench_lib is not None:
        return _bench_lib
    lib = ctypes.CDLL(_build.build("bench"))
    ci, cll, pd = ctypes.c_int, ctypes.c_longlong, ctypes.POINTER(ctypes.c_double)
    lib.hough_bench_shared_atomics.restype = ci
    lib.hough_bench_shared_atomics.argtypes = [ci, ci, ci, cll, pd]
    lib.hough_bench_vote_loop.restype = ci
    lib.hough_bench_vote_loop.argtypes = [ci, ci, ci, ci, cll, pd]
    lib.hough_bench_issue_rate.restype = ci
    lib.hough_bench_issue_rate.argtypes = [ci, ci, ci, cll, pd]
    _bench_lib = lib
    return lib


def _check(rc, what):
    if rc != HOUGH_OK:
        lib = load_library()
        raise HoughError("%s failed: %s (%s)" % (what, lib.hough_strerror(rc).decode(), lib.hough_last_error().decode()))


_dummies = {}


def _ptr(t):
    """Address of a torch tensor (None -> NULL).  torch reports a null data_ptr() for a tensor with no
    elements; the C ABI wants a real pointer for every required buffer, so an empty tensor is passed as
    the address of a small per-device scratch allocation (never read or written: there are no elements)."""
    if t is None:
        return None
    if t.numel() == 0:
        import torch
        key = (t.device.type, t.device.index)
        if key not in _dummies:
            _dummies[key] = torch.zeros(16, dtype=torch.uint8, device=t.device)
        return ctypes.c_void_p(_dummies[key].data_ptr())
    return ctypes.c_void_p(t.data_ptr())


def _stream_handle(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


# ---------------------------------------------------------------- same names as the C ABI
def hough_create(n_theta, n_rho, rho_max, threshold, window):
    lib = load_library()
    ctx = lib.hough_create(n_theta, n_rho, ctypes.c_float(rho_max), threshold, window)
    if not ctx:
        raise HoughError("hough_create failed: " + lib.hough_last_error().decode())
    return ctx


def hough_set_option(ctx, key, value):
    _check(load_library().hough_set_option(ctx, key, value), "hough_set_option")


def hough_set_option_f64(ctx, key, value):
    _check(load_library().hough_set_option_f64(ctx, key, float(value)), "hough_set_option_f64")


def _is_device_tensor(t):
    import torch
    return isinstance(t, torch.Tensor) and t.is_cuda


def hough_circles(ctx, d_xy, d_event_offsets, n_events, d_peaks, d_counts, d_circles, stream=None):
    """d_circles: CUDA uint8 tensor of at least n_events * max_peaks * 48 bytes (hough_circle records)."""
    import torch
    mp = hough_get_info(ctx, HOUGH_INFO_MAX_PEAKS)
    _marshal_check(True, n_events, d_xy, d_event_offsets, None, d_peaks, d_counts, max_peaks=mp)
    if n_events > 0 and mp > 0:
        if not (_is_device_tensor(d_circles) and d_circles.is_contiguous() and d_circles.dtype == torch.uint8
                and d_circles.numel() >= 48 * n_events * mp):
            raise HoughError("d_circles must be a contiguous CUDA uint8 tensor of at least n_events * max_peaks * 48 bytes")
    _check(load_library().hough_circles(ctx, _ptr(d_xy), _ptr(d_event_offsets), n_events, _ptr(d_peaks), _ptr(d_counts),
                                        _ptr(d_circles), _stream_handle(stream)), "hough_circles")


def hough_set_trig_table(ctx, h_cos, h_sin):
    """h_cos, h_sin: contiguous float32 numpy arrays (HOST) of n_theta entries."""
    import numpy as np
    h_cos = np.ascontiguousarray(h_cos, dtype=np.float32)
    h_sin = np.ascontiguousarray(h_sin, dtype=np.float32)
    _check(load_library().hough_set_trig_table(ctx, h_cos.ctypes.data, h_sin.ctypes.data), "hough_set_trig_table")


def hough_get_info(ctx, key):
    return int(load_library().hough_get_info(ctx, key))


def _marshal_check(cuda, n_events, xy, off, keep, peaks, counts, kept_xy=None, kept_idx=None, accum=None, max_peaks=None,
                   grid=None):
    """Marshalling-side sanity of the buffers handed to the C ABI (dtype, device, contiguity, length): the library
    itself only sees raw pointers.  No arithmetic of the method."""
    import torch
    def chk(name, t, dtype, min_numel):
        if t is None:
            return
        if not isinstance(t, torch.Tensor):
            raise HoughError("%s must be a torch tensor" % name)
        if t.dtype != dtype:
            raise HoughError("%s must be %s (got %s)" % (name, dtype, t.dtype))
        if t.is_cuda != cuda:
            raise HoughError("%s must be a %s tensor" % (name, "CUDA" if cuda else "host"))
        if not t.is_contiguous():
            raise HoughError("%s must be contiguous" % name)
        if t.numel() < min_numel:
            raise HoughError("%s holds %d elements, needs at least %d" % (name, t.numel(), min_numel))
    if n_events <= 0:
        return
    chk("event offsets", off, torch.int32, n_events + 1)
    if off is None or xy is None:
        return                         # the C ABI reports the null pointer
    n_total = xy.numel() // 2
    chk("xy", xy, torch.float32, 0)
    chk("keep mask", keep, torch.uint8, n_total)     # None (hough_circles) is skipped
    chk("counts", counts, torch.int32, 2 * n_events)
    if max_peaks:
        chk("peaks", peaks, torch.int32, 2 * n_events * max_peaks)
    chk("kept_xy", kept_xy, torch.float32, 2 * n_total)
    chk("kept_idx", kept_idx, torch.int32, n_total)
    if accum is not None and grid is not None:
        chk("accum dump", accum, torch.int32, n_events * grid[0] * grid[1])
    if cuda:
        devs = {t.device for t in (xy, off, keep, peaks, counts, kept_xy, kept_idx, accum) if t is not None and t.numel()}
        if len(devs) > 1:
            raise HoughError("all tensors must live on one device (got %s)" % sorted(map(str, devs)))


def hough_run(ctx, d_xy, d_event_offsets, n_events, d_keep_mask, d_peaks, d_counts, stream=None):
    """Tensors are CUDA torch tensors (see include/hough.h for shapes); asynchronous on `stream`."""
    _marshal_check(True, n_events, d_xy, d_event_offsets, d_keep_mask, d_peaks, d_counts,
                   max_peaks=hough_get_info(ctx, HOUGH_INFO_MAX_PEAKS))
    _check(load_library().hough_run(ctx, _ptr(d_xy), _ptr(d_event_offsets), n_events, _ptr(d_keep_mask),
                                    _ptr(d_peaks), _ptr(d_counts), _stream_handle(stream)), "hough_run")


def hough_run_ex(ctx, d_xy, d_event_offsets, n_events, d_keep_mask, d_peaks, d_counts,
                 d_kept_xy=None, d_kept_idx=None, d_accum_dump=None, stream=None):
    _marshal_check(True, n_events, d_xy, d_event_offsets, d_keep_mask, d_peaks, d_counts, d_kept_xy, d_kept_idx,
                   max_peaks=hough_get_info(ctx, HOUGH_INFO_MAX_PEAKS))
    io = hough_io(_ptr(d_xy), _ptr(d_event_offsets), n_events, _ptr(d_keep_mask), _ptr(d_peaks), _ptr(d_counts),
                  _ptr(d_kept_xy), _ptr(d_kept_idx), _ptr(d_accum_dump))
    _check(load_library().hough_run_ex(ctx, ctypes.byref(io), _stream_handle(stream)), "hough_run_ex")


def hough_run_host(ctx, h_xy, h_event_offsets, n_events, h_keep_mask, h_peaks, h_counts,
                   h_kept_xy=None, h_kept_idx=None, stream=None):
    """HOST (ideally pinned) torch tensors in and out; copies are inside the call, asynchronous on `stream`."""
    _marshal_check(False, n_events, h_xy, h_event_offsets, h_keep_mask, h_peaks, h_counts, h_kept_xy, h_kept_idx,
                   max_peaks=hough_get_info(ctx, HOUGH_INFO_MAX_PEAKS))
    _check(load_library().hough_run_host(ctx, _ptr(h_xy), _ptr(h_event_offsets), n_events, _ptr(h_keep_mask),
                                         _ptr(h_peaks), _ptr(h_counts), _ptr(h_kept_xy), _ptr(h_kept_idx),
                                         _stream_handle(stream)), "hough_run_host")


def hough_destroy(ctx):
    load_library().hough_destroy(ctx)


def hough_version():
    return load_library().hough_version().decode()


def _bench_call(name, *args):
    out = ctypes.c_double(0.0)
    rc = getattr(load_bench_library(), name)(*args, ctypes.byref(out))
    if rc != 0:
        raise HoughError("%s failed with status %d%s" % (name, rc, " (no CUDA device?)" if rc == -3 else ""))
    return out.value


def hough_bench_shared_atomics(variant, ctas_per_sm, threads, iters):
    """Shared atomics per second over the whole device (include/hough_bench.h); variant 5 = the roofline's peak."""
    return _bench_call("hough_bench_shared_atomics", variant, ctas_per_sm, threads, iters)


def hough_bench_vote_loop(mode, cpl, ctas_per_sm, threads, iters):
    """Lane-votes per second of the voting loop's instruction mix (include/hough_bench.h)."""
    return _bench_call("hough_bench_vote_loop", mode, cpl, ctas_per_sm, threads, iters)


def hough_bench_issue_rate(kind, ctas_per_sm, threads, iters):
    """Warp-instructions per second of one instruction class (include/hough_bench.h)."""
    return _bench_call("hough_bench_issue_rate", kind, ctas_per_sm, threads, iters)


def hough_debug_tame_bounds(n_rho, rho_max, table_max, table_min_nz):
    """(tame_bound, ftz_min) as the kernel receives them (include/hough_debug.h); host-only."""
    out = (ctypes.c_float * 2)()
    _check(load_library().hough_debug_tame_bounds(n_rho, ctypes.c_float(rho_max), ctypes.c_float(table_max),
                                                  ctypes.c_float(table_min_nz), out), "hough_debug_tame_bounds")
    return float(out[0]), float(out[1])


def hough_debug_bounds_enabled():
    return bool(load_library().hough_debug_bounds_enabled())


PLAN_FIELDS = ("cluster_size", "threads", "smem_bytes", "acc_bits", "cols_per_lane", "cols_per_cta", "n_groups", "n_stripes",
               "pitch_bytes", "bitmap_words_per_row", "chunk_hits", "region_bytes", "pbm_off", "pbm_bytes", "hb_off", "misc_off",
               "w8_off", "w8_pitch", "mcf_off", "msf_off", "colq_off", "stash_off", "cnt_off", "gcnt_off", "rcp_groups", "rcp_2s", "circ_cap")


def hough_plan_describe(n_theta, n_rho, acc_dtype=HOUGH_ACC_AUTO, cluster_size=0, ctas_per_sm=0, smem_optin=0):
    """Launch shape and shared-memory layout the library would choose (host-only, needs no GPU) as a dict."""
    out = (ctypes.c_longlong * len(PLAN_FIELDS))()
    _check(load_library().hough_plan_describe(n_theta, n_rho, acc_dtype, cluster_size, ctas_per_sm, smem_optin, out, len(PLAN_FIELDS)),
           "hough_plan_describe")
    return dict(zip(PLAN_FIELDS, [int(x) for x in out]))


# ---------------------------------------------------------------- convenience wrapper (allocation + marshalling only)
class Hough:
    """Owns a hough_ctx and allocates output tensors.  No arithmetic of the method happens here."""

    def __init__(self, n_theta, n_rho, rho_max, threshold, window, max_peaks=64, acc_dtype="u16",
                 conformal_scale=1, cluster_size=0, ctas_per_sm=0, trig_table=None, peak_mode=0, rel_permille=500,
                 nms_radius=1, theta_wrap=False, keep_mode=0, keep_tol=0.0, b_field=1.0, staging=0, scheduler=0, select_mode=0):
        self.n_theta, self.n_rho, self.max_peaks = n_theta, n_rho, max_peaks
        self.ctx = hough_create(n_theta, n_rho, float(rho_max), threshold, window)
        try:
            hough_set_option(self.ctx, HOUGH_OPT_MAX_PEAKS, max_peaks)
            hough_set_option(self.ctx, HOUGH_OPT_ACC_DTYPE, {"auto": 0, "u16": 1, "u32": 2}[acc_dtype])
            if conformal_scale != 1:
                hough_set_option(self.ctx, HOUGH_OPT_CONFORMAL_SCALE, conformal_scale)
            if cluster_size:
                hough_set_option(self.ctx, HOUGH_OPT_CLUSTER_SIZE, cluster_size)
            if ctas_per_sm:
                hough_set_option(self.ctx, HOUGH_OPT_CTAS_PER_SM, ctas_per_sm)
            if trig_table is not None:
                hough_set_trig_table(self.ctx, trig_table[0], trig_table[1])
            if peak_mode:
                hough_set_option(self.ctx, HOUGH_OPT_PEAK_MODE, peak_mode)
                hough_set_option(self.ctx, HOUGH_OPT_REL_THRESHOLD_PERMILLE, rel_permille)
                hough_set_option(self.ctx, HOUGH_OPT_NMS_RADIUS, nms_radius)
            if theta_wrap:
                hough_set_option(self.ctx, HOUGH_OPT_THETA_WRAP, 1)
            if keep_mode:
                hough_set_option(self.ctx, HOUGH_OPT_KEEP_MODE, keep_mode)
                hough_set_option_f64(self.ctx, HOUGH_OPTF_KEEP_TOL, keep_tol)
            if b_field != 1.0:
                hough_set_option_f64(self.ctx, HOUGH_OPTF_B_FIELD_TESLA, b_field)
            if staging:
                hough_set_option(self.ctx, HOUGH_OPT_STAGING, staging)
            if scheduler:
                hough_set_option(self.ctx, HOUGH_OPT_SCHEDULER, scheduler)
            if select_mode:
                hough_set_option(self.ctx, HOUGH_OPT_SELECT_MODE, select_mode)
        except Exception:
            self.close()
            raise

    def info(self, key):
        return hough_get_info(self.ctx, key)

    def alloc_outputs(self, n_total, n_events, device="cuda", kept=True, accum=False):
        import torch
        out = {
            "keep": torch.zeros(max(n_total, 1), dtype=torch.uint8, device=device)[:n_total],
            "peaks": torch.zeros((n_events, max(self.max_peaks, 1), 2), dtype=torch.int32, device=device)[:, :self.max_peaks],
            "counts": torch.zeros((n_events, 2), dtype=torch.int32, device=device),
        }
        if kept:
            out["kept_xy"] = torch.zeros((max(n_total, 1), 2), dtype=torch.float32, device=device)[:n_total]
            out["kept_idx"] = torch.zeros(max(n_total, 1), dtype=torch.int32, device=device)[:n_total]
        if accum:
            out["accum"] = torch.zeros((n_events, self.n_theta, self.n_rho), dtype=torch.int32, device=device)
        return out

    def run(self, d_xy, d_offsets, out=None, stream=None, kept=True, accum=False):
        """d_xy [N,2] f32 cuda, d_offsets [n_events+1] i32 cuda.  Returns the dict of output tensors
        (peaks as int32 [n_events, max_peaks, 2]: word 0 = theta_bin | rho_bin << 16, word 1 = votes)."""
        n_events = d_offsets.numel() - 1
        n_total = d_xy.shape[0]
        if out is None:
            out = self.alloc_outputs(n_total, n_events, d_xy.device, kept=kept, accum=accum)
        hough_run_ex(self.ctx, d_xy, d_offsets, n_events, out["keep"], out["peaks"], out["counts"],
                     out.get("kept_xy"), out.get("kept_idx"), out.get("accum"), stream)
        return out

    def circles(self, d_xy, d_offsets, out, stream=None):
        """Candidate circles of the stored peaks of `out` (the dict run() returned): a CUDA uint8 tensor
        [n_events, max_peaks, 48] of hough_circle records (view it with CIRCLE_DTYPE on the host)."""
        import torch
        n_events = d_offsets.numel() - 1
        circ = torch.zeros((n_events, max(self.max_peaks, 1), 48), dtype=torch.uint8, device=d_xy.device)[:, :self.max_peaks]
        hough_circles(self.ctx, d_xy, d_offsets, n_events, out["peaks"], out["counts"], circ, stream)
        return circ

    def close(self):
        if getattr(self, "ctx", None):
            hough_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def circle_dtype():
    """numpy dtype of hough_circle (include/hough.h): pure layout, for viewing the bytes hough_circles wrote."""
    import numpy as np
    return np.dtype([("x_c", "<f8"), ("y_c", "<f8"), ("r_c", "<f8"), ("pt", "<f8"), ("phi0", "<f8"), ("charge", "<i4"), ("n_hits", "<i4")])


def unpack_peaks(peaks_i32):
    """[n_events, max_peaks, 2] int32 (torch or numpy, on the host) -> numpy [n_events, max_peaks, 3] u32
    (theta_bin, rho_bin, votes).  Pure bit unpacking of the hough_peak struct."""
    import numpy as np
    a = np.ascontiguousarray(peaks_i32.cpu().numpy() if hasattr(peaks_i32, "cpu") else peaks_i32).view(np.uint32)
    out = np.empty(a.shape[:2] + (3,), dtype=np.uint32)
    out[..., 0] = a[..., 0] & 0xFFFF
    out[..., 1] = a[..., 0] >> 16
    out[..., 2] = a[..., 1]
    return out
