"""The product's HOST code without a GPU (tests/simt_emu/host.py): paper_2607_04067_b200/csrc/hough_api.cu -- handles,
options, planner, launch set-up, hough_run_host's staging areas and pointer arithmetic -- compiled by g++ against a fake
CUDA runtime whose "device" memory ends at guard pages and whose kernel launches run the kernel source under the SIMT
emulator.  The same entry points a GPU user calls, numpy arrays for device buffers, results against the oracle.  This
is what tests/test_kernel_emulation.py does for the kernel alone, extended to the code in front of it (which round 2
rewrote and could not run on a GPU).  Not a parity claim for the device code: only `-m gpu` tests are."""
import os
import sys

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)
sys.path.insert(0, os.path.dirname(HERE))

import oracle  # noqa: E402
import paper_2607_04067_b200 as hb  # noqa: E402
import stcf_inputs as si  # noqa: E402
from simt_emu import host  # noqa: E402
from test_parity_gpu import compare  # noqa: E402


def in_child(fn):
    """Runs the test in a forked child: the emulator ends the process when it finds a fault (a guard page, a failed check
    of simt_shim.h), and that must fail one test, not end the pytest run."""
    import functools
    import traceback

    @functools.wraps(fn)
    def wrapper(*a, **k):
        r, wfd = os.pipe()
        sys.stdout.flush(); sys.stderr.flush()
        pid = os.fork()
        if pid == 0:
            os.close(r)
            code = 0
            try:
                fn(*a, **k)
            except BaseException:  # noqa: BLE001
                os.write(wfd, traceback.format_exc().encode()[-6000:])
                code = 1
            sys.stdout.flush(); sys.stderr.flush()
            os._exit(code)
        os.close(wfd)
        text = b""
        while True:
            chunk = os.read(r, 65536)
            if not chunk:
                break
            text += chunk
        os.close(r)
        _, status = os.waitpid(pid, 0)
        if status != 0:
            pytest.fail("in the child process (wait status %d):\n%s" % (status, text.decode(errors="replace")), pytrace=False)
    return wrapper


def make(cfg, **kw):
    w = si.config(cfg)
    table = si.trig_table(w.n_theta)
    base = dict(max_peaks=w.max_peaks, acc_dtype=w.acc_dtype)
    base.update(kw)
    return w, table, host.Handle(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table, **base)


def reference(w, table, xy, off, accum=False, **kw):
    return oracle.run(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table[0], table[1], max_peaks=kw.get("max_peaks", w.max_peaks),
                      acc_u16=kw.get("acc_dtype", w.acc_dtype) != "u32", want_accum=accum)


def host_outputs(n_total, n_ev, max_peaks, poison=True):
    return dict(keep=np.full(n_total, 7 if poison else 0, np.uint8), peaks=np.full((n_ev, max_peaks, 2), -1, np.int32),
                counts=np.full((n_ev, 2), -99, np.int32), kept_xy=np.full((n_total, 2), 3.0, np.float32), kept_idx=np.full(n_total, -5, np.int32))


def check_host_result(g, o, off, max_peaks, e0=0, lean=False):
    """hough_run_host's contract: the entries hough_run defines equal the oracle's, the rest of h_peaks and of the kept
    arrays (of the sub-batch's own hits) is zero."""
    n_ev = len(off) - 1
    assert np.array_equal(g["counts"], o.counts[e0:e0 + n_ev])
    lo, hi = int(off[0]), int(off[-1])
    assert np.array_equal(g["keep"][lo:hi], o.keep[lo:hi])
    p3 = hb.unpack_peaks(g["peaks"])
    for e in range(n_ev):
        ns = min(int(o.counts[e0 + e, 0]), max_peaks)
        assert np.array_equal(p3[e, :ns], o.peaks[e0 + e, :ns]), "peaks of event %d" % (e0 + e)
        assert not g["peaks"][e, ns:].any(), "peak tail of event %d is not zero" % (e0 + e)
        if lean:
            continue
        a, b, nk = int(off[e]), int(off[e + 1]), int(o.counts[e0 + e, 1])
        assert np.array_equal(g["kept_idx"][a:a + nk], o.kept_idx[a:a + nk])
        assert np.array_equal(g["kept_xy"][a:a + nk].view(np.uint32), o.kept_xy[a:a + nk].view(np.uint32))
        assert not g["kept_idx"][a + nk:b].any() and not g["kept_xy"][a + nk:b].any(), "kept tail of event %d is not zero" % (e0 + e)


@in_child
def test_run_ex_through_the_real_host_code_matches_the_oracle_and_nothing_leaks():
    w, table, h = make(0)
    before = host.counters(h.lib)
    xy, off, _ = si.generate(w, 3)
    g = h.run(xy, off, accum=True)
    g["peaks3"] = hb.unpack_peaks(g["peaks"])
    compare(g, reference(w, table, xy, off, accum=True), off, w.max_peaks, accum=True, tag="host emulation")
    assert h.info(hb.HOUGH_INFO_LAUNCHES) == 1 and host.counters(h.lib)["launches"] == before["launches"] + 1
    assert host.counters(h.lib)["malloc"] == before["malloc"], "hough_run_ex allocated device memory"
    h.close()
    c = host.counters(h.lib)
    assert c["malloc"] == c["free"], "hough_destroy left device allocations behind"


@pytest.mark.parametrize("lean", [False, True])
@in_child
def test_run_host_whole_batch(lean):
    w, table, h = make(0)
    xy, off, _ = si.generate(w, 4)
    o = reference(w, table, xy, off)
    g = host_outputs(len(xy), 4, w.max_peaks)
    h.run_host(xy, off, 4, g["keep"], g["peaks"], g["counts"], None if lean else g["kept_xy"], None if lean else g["kept_idx"])
    check_host_result(g, o, off, w.max_peaks, lean=lean)
    if lean:
        assert (g["kept_idx"] == -5).all()                   # never touched
    h.close()
    c = host.counters(h.lib)
    assert c["malloc"] == c["free"]


@pytest.mark.parametrize("staging", [0, 1])
@in_child
def test_run_host_sub_batches_with_absolute_offsets_on_many_streams(staging):
    """Sub-batches of one host array: the same array pointers, the offsets advanced to the sub-batch's first event, one
    staging area per stream, 10 streams on 8 slots (the least recently used slot is recycled).  The first hit of a
    sub-batch may sit at an odd index: the staged copy keeps its 16-byte phase (bulk-copy staging relies on it)."""
    w, table, h = make(0, staging=staging)
    xy, off, _ = si.generate(w, 11)
    if not (off[1:-1] & 1).any():                            # make sure an odd first hit occurs
        xy, off = xy[1:], off.copy()
        off[1:] -= 1
    assert (off[1:-1] & 1).any()
    o = reference(w, table, xy, off)
    keep = np.full(len(xy), 7, np.uint8)
    kxy, kidx = np.full((len(xy), 2), 3.0, np.float32), np.full(len(xy), -5, np.int32)
    cuts = [0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11]
    for rnd in range(2):                                     # the second round re-uses (and recycles) the slots
        for b, (e0, e1) in enumerate(zip(cuts[:-1], cuts[1:])):
            n_ev = e1 - e0
            peaks, counts = np.full((n_ev, w.max_peaks, 2), -1, np.int32), np.full((n_ev, 2), -99, np.int32)
            h.run_host(xy, off[e0:], n_ev, keep, peaks, counts, kxy, kidx, stream=1 + (b % 10) + 16 * rnd)
            check_host_result(dict(keep=keep, peaks=peaks, counts=counts, kept_xy=kxy, kept_idx=kidx), o, off[e0:e1 + 1], w.max_peaks, e0=e0)
    assert np.array_equal(keep, o.keep)                      # every hit of the array was covered exactly by its own sub-batch
    h.close()
    c = host.counters(h.lib)
    assert c["malloc"] == c["free"]


@in_child
def test_run_host_grows_its_staging_area_and_handles_empty_batches():
    w, table, h = make(0)
    xy, off, _ = si.generate(w, 6)
    o = reference(w, table, xy, off)
    for n_ev in (1, 6, 2):                                   # grow, then a smaller batch in the grown area
        g = host_outputs(len(xy), n_ev, w.max_peaks)
        h.run_host(xy, off, n_ev, g["keep"], g["peaks"], g["counts"], g["kept_xy"], g["kept_idx"], stream=5)
        check_host_result(g, o, off[:n_ev + 1], w.max_peaks)
    # events without hits, and a batch of only such events
    off0 = np.zeros(4, np.int32)
    g = host_outputs(0, 3, w.max_peaks)
    h.run_host(np.zeros((0, 2), np.float32), off0, 3, g["keep"], g["peaks"], g["counts"], g["kept_xy"], g["kept_idx"], stream=5)
    assert (g["counts"] == 0).all() and not g["peaks"].any()
    h.close()


@in_child
def test_two_live_handles_of_one_instantiation_with_different_footprints():
    """cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel, not to a handle: it is only ever raised (the
    fake runtime refuses a launch whose shared memory exceeds the attribute, as the real one does)."""
    w = si.config(0)
    small = host.Handle(180, 128, w.rho_max, w.threshold, w.window, si.trig_table(180), max_peaks=16)
    big = host.Handle(180, 256, w.rho_max, w.threshold, w.window, si.trig_table(180), max_peaks=16)
    assert small.info(hb.HOUGH_INFO_SMEM_BYTES) < big.info(hb.HOUGH_INFO_SMEM_BYTES)
    xy, off, _ = si.generate(w, 2)
    for h, nr in ((big, 256), (small, 128), (big, 256)):
        g = h.run(xy, off)
        o = oracle.run(xy, off, 180, nr, w.rho_max, w.threshold, w.window, *si.trig_table(180), max_peaks=16, acc_u16=True)
        assert np.array_equal(g["counts"], o.counts) and np.array_equal(g["keep"], o.keep)
    small.close(); big.close()


@in_child
def test_circles_and_every_option_through_the_abi():
    w = si.config(1)
    table = si.trig_table(w.n_theta)
    opts = dict(peak_mode=1, rel_permille=400, nms_radius=2, theta_wrap=True, keep_mode=1, keep_tol=5.0)
    h = host.Handle(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table, max_peaks=w.max_peaks, acc_dtype=w.acc_dtype,
                    cluster_size=2, staging=1, b_field=1.0, **opts)
    xy, off, _ = si.generate(w, 2)
    g = h.run(xy, off)
    # the variants that change nothing: dense selection + work stealing on a one-CTA-per-event grid, through set_option
    hv = host.Handle(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table, max_peaks=w.max_peaks, acc_dtype=w.acc_dtype,
                     select_mode=1, scheduler=1, staging=1)
    gv, gd = hv.run(xy, off), host.Handle(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table, max_peaks=w.max_peaks).run(xy, off)
    assert all(np.array_equal(gv[k], gd[k]) for k in ("keep", "counts", "peaks", "kept_idx"))
    assert hv.lib.hough_set_option(hv.ctx, hb.HOUGH_OPT_SELECT_MODE, 3) != hb.HOUGH_OK
    hv.close()
    circ = h.circles(xy, off, g)
    o, oc = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table[0], table[1], max_peaks=w.max_peaks,
                          acc_u16=True, want_circles=True, n_threads=4, **opts)
    g["peaks3"] = hb.unpack_peaks(g["peaks"])
    compare(g, o, off, w.max_peaks, accum=False, tag="ext")
    for e in range(2):
        ns = min(int(o.counts[e, 0]), w.max_peaks)
        assert circ[e, :ns].tobytes() == oc[e, :ns].tobytes()
    h.close()


@in_child
def test_refusals_of_the_host_code():
    w, table, h = make(0)
    assert h.lib.hough_set_option(h.ctx, hb.HOUGH_OPT_VOTE_PATH, 2) != hb.HOUGH_OK          # the diagnostics are not in this build
    assert h.lib.hough_set_option(h.ctx, 99, 0) != hb.HOUGH_OK
    assert h.lib.hough_set_option(h.ctx, hb.HOUGH_OPT_CLUSTER_SIZE, 3) != hb.HOUGH_OK
    xy, off, _ = si.generate(w, 1)
    g = h.outputs(len(xy), 1)
    io = hb.hough_io(None, off.ctypes.data, 1, g["keep"].ctypes.data, g["peaks"].ctypes.data, g["counts"].ctypes.data, None, None, None)
    import ctypes
    assert h.lib.hough_run_ex(h.ctx, ctypes.byref(io), None) != hb.HOUGH_OK and b"" != h.lib.hough_last_error()
    assert host.counters(h.lib)["launches"] >= 0
    h.close()
    assert hb.hough_create is not None and not h.lib.hough_create(0, 256, 0.003, 16, 1)         # bad grid: NULL handle


@in_child
def test_run_host_under_the_race_and_init_check():
    """The race-check build of the same library: every byte the kernel reads was written by a copy, a memset or the
    kernel itself (an initcheck of hough_run_host's staging), and no launch races."""
    w, table, h = make(1, race=True, staging=1)
    xy, off, _ = si.generate(w, 3)
    o = reference(w, table, xy, off)
    g = host_outputs(len(xy), 2, w.max_peaks)
    h.run_host(xy, off[1:], 2, g["keep"], g["peaks"], g["counts"], g["kept_xy"], g["kept_idx"], stream=3)
    check_host_result(g, o, off[1:], w.max_peaks, e0=1)
    circ = h.circles(xy, off, h.run(xy, off))
    assert host.counters(h.lib)["reports"] == 0
    h.close()
