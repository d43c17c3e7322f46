"""-m "not gpu": the CUDA kernel's own source, compiled for the CPU under a SIMT emulator (tests/simt_emu), against
the oracle -- accumulators, peak lists, counts, keep masks, compacted order -- on small seeded inputs.  This checks
the kernel's LOGIC without a GPU (indexing, phase order, shared-memory layout, bounds: every buffer ends at a guard
page, and the debug-bounds flavour must report no violation); it is not the parity gate -- the `-m gpu` tests are."""
import numpy as np
import pytest

import oracle
import stcf_inputs as si
from tests import simt_emu
from tests.test_parity_gpu import compare


def emu_both(w, xy, off, accum=True, **kw):
    table = si.trig_table(w.n_theta)
    args = dict(max_peaks=w.max_peaks, acc_dtype=w.acc_dtype, threshold=w.threshold, window=w.window)
    args.update(kw)
    emu_only = {k: args.pop(k) for k in ("cluster_size", "ctas_per_sm", "vote_path", "grid_clusters", "debug_bounds", "order") if k in args}
    g = simt_emu.run(xy, off, w.n_theta, w.n_rho, w.rho_max, args["threshold"], args["window"], table,
                     max_peaks=args["max_peaks"], acc_dtype=args["acc_dtype"], accum=accum,
                     conformal_scale=args.get("conformal_scale", 1), **emu_only)
    o = oracle.run(xy, off, w.n_theta, w.n_rho, w.rho_max, args["threshold"], args["window"], table[0], table[1],
                   max_peaks=args["max_peaks"], conformal_scale=args.get("conformal_scale", 1),
                   acc_u16=(args["acc_dtype"] != "u32"), want_accum=accum, n_threads=4)
    assert not np.any(g["counts"][:, 0] == -2), "debug-bounds sentinel: phases %s" % g["counts"][g["counts"][:, 0] == -2, 1]
    compare(g, o, off, args["max_peaks"], accum=accum, tag=w.name)
    return g, o


def test_w1_worked_example_under_the_emulator():
    xy = np.array([[1, 0], [0, 1], [.5, .5], [-1, 0], [0, 0], [4, 0]], dtype=np.float32)
    off = np.array([0, 6], dtype=np.int32)
    table = si.trig_table(4)
    for thr, w, exp_keep in ((2, 0, [1, 1, 1, 1, 0, 1]), (3, 0, [1, 0, 0, 1, 0, 1]), (3, 1, [1, 1, 1, 1, 0, 1])):
        g = simt_emu.run(xy, off, 4, 8, 2.0, thr, w, table, max_peaks=8)
        o = oracle.run(xy, off, 4, 8, 2.0, thr, w, table[0], table[1], max_peaks=8, want_accum=True)
        compare(g, o, off, 8, tag="W1")
        assert g["keep"].tolist() == exp_keep


@pytest.mark.parametrize("cfg,n_ev,dbg", [(0, 3, False), (0, 2, True), (1, 2, True), (2, 1, True), (3, 1, True)])
def test_configs_under_the_emulator(cfg, n_ev, dbg):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    emu_both(w, xy, off, debug_bounds=dbg)


@pytest.mark.parametrize("cluster", [2, 8])
def test_clusters_under_the_emulator(cluster):
    w = si.config(0)
    xy, off, _ = si.generate(w, 2)
    g, _ = emu_both(w, xy, off, cluster_size=cluster, debug_bounds=True)
    assert g["info"]["CLUSTER_SIZE"] == cluster


def test_cluster_grid_360x512_under_the_emulator():
    w = si.config(5)
    xy, off, _ = si.generate(w, 1)
    g, _ = emu_both(w, xy, off, debug_bounds=True)
    assert g["info"]["CLUSTER_SIZE"] == 2


def test_event_loop_empty_events_and_degenerate_hits_under_the_emulator():
    w = si.config(0)
    xy, off, _ = si.generate(w, 3)
    bad = np.array([[0, 0], [np.inf, 1], [1e-3, 0], [1e-20, 1e-20], [np.nan, 5], [1e30, 1e30], [3e38, 0]], dtype=np.float32)
    xy2 = np.concatenate([xy[:off[1]], bad, xy[off[1]:]])
    off2 = np.concatenate([[0, 0], off[1:2] + len(bad), off[2:] + len(bad), [off[-1] + len(bad)]]).astype(np.int32)
    emu_both(w, xy2, off2, threshold=5, grid_clusters=2, debug_bounds=True)     # 5 events on 2 CTAs: the event loop iterates
    emu_both(w, xy2, off2, threshold=5, vote_path=1)


def test_truncation_and_window_under_the_emulator():
    w = si.config(2)
    xy, off, _ = si.generate(w, 1)
    emu_both(w, xy, off, max_peaks=3, window=2, debug_bounds=True)
    emu_both(w, xy, off, max_peaks=0)


# ---------------------------------------------------------------- the NEXT rows under the emulator (against oracle.run_ex)
def emu_ex(w, xy, off, accum=True, circles=False, **kw):
    table = si.trig_table(w.n_theta)
    base = dict(max_peaks=w.max_peaks, acc_dtype=w.acc_dtype, threshold=w.threshold, window=w.window, conformal_scale=1)
    base.update({k: kw.pop(k) for k in list(kw) if k in base})
    opts = {k: kw.pop(k) for k in list(kw) if k in ("peak_mode", "rel_permille", "nms_radius", "theta_wrap", "keep_mode", "keep_tol", "b_field")}
    emu_only = {k: kw.pop(k) for k in list(kw) if k in ("staging", "order", "scheduler", "steals", "select_mode")}
    rho_max = kw.pop("rho_max", w.rho_max)
    g = simt_emu.run(xy, off, w.n_theta, w.n_rho, rho_max, base["threshold"], base["window"], table, max_peaks=base["max_peaks"],
                     acc_dtype=base["acc_dtype"], accum=accum, conformal_scale=base["conformal_scale"], circles=circles, **opts, **emu_only, **kw)
    o, oc = oracle.run_ex(xy, off, w.n_theta, w.n_rho, rho_max, base["threshold"], base["window"], table[0], table[1],
                          max_peaks=base["max_peaks"], conformal_scale=base["conformal_scale"], acc_u16=(base["acc_dtype"] != "u32"),
                          want_accum=accum, n_threads=4, want_circles=circles, **opts)
    assert not np.any(g["counts"][:, 0] == -2), "debug-bounds sentinel: phases %s" % g["counts"][g["counts"][:, 0] == -2, 1]
    compare(g, o, off, base["max_peaks"], accum=accum, tag=w.name)
    if circles:
        for e in range(len(off) - 1):
            ns = min(int(o.counts[e, 0]), base["max_peaks"])
            assert g["circles"][e, :ns].tobytes() == oc[e, :ns].tobytes(), "circles of event %d" % e     # bit for bit, fp64 included
            assert np.all(np.frombuffer(g["circles"][e, ns:].tobytes(), dtype=np.uint8) == 0xFF)           # the rest is untouched
    return g, o


def test_n1_circles_under_the_emulator():
    w = si.config(0)
    xy, off, _ = si.generate(w, 3)
    emu_ex(w, xy, off, circles=True, debug_bounds=True, b_field=1.0)
    emu_ex(w, xy, off, circles=True, conformal_scale=2, rho_max=float(np.float32(2) * np.float32(w.rho_max)), b_field=0.8)
    w1 = si.config(0, 1)
    w1 = type(w1)(**{**w1.__dict__, "n_theta": 4, "n_rho": 8, "rho_max": 2.0, "threshold": 2, "window": 0, "max_peaks": 8})
    xy1 = np.array([[1, 0], [0, 1], [.5, .5], [-1, 0], [0, 0], [4, 0]], dtype=np.float32)
    g, _ = emu_ex(w1, xy1, np.array([0, 6], dtype=np.int32), circles=True)
    assert [int(c) for c in g["circles"][0, :3]["charge"]] == [-1, -1, 1] and g["circles"][0, 2]["r_c"] == 2.0     # tests/golden/w1_next.txt


@pytest.mark.parametrize("cfg,permille,radius,wrap", [(0, 500, 1, False), (1, 300, 2, False), (0, 0, 0, True), (3, 600, 3, True)])
def test_n2_iterative_nms_under_the_emulator(cfg, permille, radius, wrap):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, 2 if cfg != 3 else 1)
    g, o = emu_ex(w, xy, off, peak_mode=1, rel_permille=permille, nms_radius=radius, theta_wrap=wrap, debug_bounds=True)
    assert o.counts[:, 0].min() >= 1
    emu_ex(w, xy, off, peak_mode=1, rel_permille=permille, nms_radius=radius, theta_wrap=wrap, max_peaks=2)


@pytest.mark.parametrize("cluster,window", [(0, 1), (0, 3), (2, 2)])
def test_n4a_theta_wrap_under_the_emulator(cluster, window):
    w = si.config(0)
    xy, off, _ = si.generate(w, 3)
    # a noiseless track whose centre direction (179.8 deg) sits on the theta seam: it peaks at column 0 AND, mirrored, at 179
    r = 200.0 + np.arange(48) * 600.0 / 47.0
    phi = np.deg2rad(179.8) - np.arccos(r / 1200.0)
    xy = np.concatenate([np.stack([r * np.cos(phi), r * np.sin(phi)], axis=1).astype(np.float32), xy])
    off = off.copy()
    off[1:] += 48
    g, o = emu_ex(w, xy, off, theta_wrap=True, window=window, threshold=12, max_peaks=512, cluster_size=cluster, debug_bounds=True)
    o0, _ = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, 12, window, *si.trig_table(w.n_theta), max_peaks=512)
    assert not np.array_equal(o.keep, o0.keep) or not np.array_equal(o.counts, o0.counts)      # the seam matters on these events


@pytest.mark.parametrize("cluster,tol", [(0, 5.0), (2, 20.0), (0, 0.0)])
def test_n4b_distance_filter_under_the_emulator(cluster, tol):
    w = si.config(0)
    xy, off, _ = si.generate(w, 3)
    emu_ex(w, xy, off, keep_mode=1, keep_tol=tol, cluster_size=cluster, debug_bounds=True)


def test_n3_the_papers_1000x1000_grid_under_the_emulator():
    # rho in [-0.01, 0.01] and theta in [0, pi), 1000 bins each; 0.01/mm = 2/r at r = 200 mm, i.e. the scale
    # of Eq. (2).  2 MB of u16 cells: a 16-CTA (non-portable) cluster, 63 theta columns per CTA
    w = si.config(0)
    w = type(w)(**{**w.__dict__, "n_theta": 1000, "n_rho": 1000, "rho_max": 0.01, "threshold": 12, "window": 2, "max_peaks": 64})
    xy, off, _ = si.generate(w, 1)
    g, o = emu_ex(w, xy, off, conformal_scale=2, debug_bounds=True, accum=True)
    assert g["info"]["CLUSTER_SIZE"] == 16 and o.counts[0, 0] >= 2


# ---------------------------------------------------------------- scheduling-order independence (a weak synccheck)
@pytest.mark.parametrize("order", ["reverse", "shuffle:1", "shuffle:2"])
def test_results_do_not_depend_on_the_order_in_which_threads_reach_their_barriers(order):
    # a fiber runs until its next barrier / warp collective; a phase that reads what another thread has not yet written
    # (a missing barrier) gives different results when the threads take their turns in another order
    w = si.config(0)
    xy, off, _ = si.generate(w, 2)
    emu_both(w, xy, off, order=order)
    emu_both(w, xy, off, cluster_size=2, order=order)
    w1 = si.config(1)
    xy1, off1, _ = si.generate(w1, 1)
    emu_ex(w1, xy1, off1, peak_mode=1, rel_permille=300, nms_radius=2, circles=True, order=order)
    emu_ex(w, xy, off, theta_wrap=True, keep_mode=1, keep_tol=5.0, cluster_size=2, order=order)
    w3 = si.config(3)
    xy3, off3, _ = si.generate(w3, 4)
    big = np.ascontiguousarray(xy3[:off3[4]])          # ~11000 hits as one event: several staging chunks, several selection blocks
    emu_both(w3, big, np.array([0, len(big)], dtype=np.int32), threshold=45, cluster_size=2, order=order)


# ---------------------------------------------------------------- bulk-copy staging (HOUGH_OPT_STAGING = 1) under the emulator
@pytest.mark.parametrize("cfg,n_ev,cluster", [(0, 5, 0), (1, 3, 0), (0, 4, 2), (3, 2, 0)])
def test_bulk_copy_staging_under_the_emulator(cfg, n_ev, cluster):
    # events start at odd and even hit indices; the emulator checks every copy: 16-byte aligned source, destination and
    # size, source inside the hit array (the batch's odd last hit must come from a plain load)
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    emu_ex(w, xy, off, staging=1, cluster_size=cluster, debug_bounds=True)
    # without the batch's first hit every later event starts at the other parity, and the batch ends on the other parity
    off2 = np.concatenate([[0], off[1:] - 1]).astype(np.int32)
    emu_ex(w, xy[1:], off2, staging=1, cluster_size=cluster, debug_bounds=True)
    assert {int(o) & 1 for o in off[1:-1]} | {int(o) & 1 for o in off2[1:-1]} == {0, 1} and (len(xy) - 1) % 2 != len(xy) % 2


def test_bulk_copy_staging_edge_cases_under_the_emulator():
    w = si.config(0)
    xy, off, _ = si.generate(w, 3)
    # empty events, one-hit and two-hit events, the last event a single (odd) hit
    xy1 = np.concatenate([xy[:off[1]], np.array([[300, 0], [0, 450], [200, 200], [-700, 100]], dtype=np.float32)])
    off1 = np.array([0, 0, off[1], off[1] + 1, off[1] + 3, off[1] + 3, off[1] + 4], dtype=np.int32)
    emu_ex(w, xy1, off1, staging=1, threshold=1, max_peaks=512, debug_bounds=True)
    # an event larger than the staging chunk: several copies per event, every chunk with its own alignment shift
    w3 = si.config(3)
    xy3, off3, _ = si.generate(w3, 4)
    big = np.ascontiguousarray(xy3[1:off3[4]])
    emu_ex(w3, big, np.array([0, 5, len(big)], dtype=np.int32), staging=1, threshold=45, debug_bounds=True)
    emu_ex(w3, big, np.array([0, 5, len(big)], dtype=np.int32), staging=1, threshold=45, cluster_size=2, acc_dtype="u16", order="shuffle:3")
    # together with the other options of the extended instantiation
    emu_ex(w, xy, off, staging=1, peak_mode=1, theta_wrap=True, keep_mode=1, keep_tol=5.0, circles=True)


# ---------------------------------------------------------------- work-stealing scheduler (HOUGH_OPT_SCHEDULER = 1) under the emulator
@pytest.mark.parametrize("steals", [None, 0, 1, 3])
def test_work_stealing_scheduler_under_the_emulator(steals):
    # the emulator runs one CTA after the other and hands a running CTA's cancellation requests the not-yet-launched
    # CTAs: without a limit the first CTA takes over every event; steals = 0 makes every request fail (one event per CTA,
    # as without the option); small limits mix stolen and regularly launched CTAs.  Every event must come out exactly
    # once and bit-identical, empty / refused / chunked events included.
    w = si.config(0)
    xy, off, _ = si.generate(w, 7)
    off2 = np.concatenate([[0, 0], off[1:4], [off[3]], off[4:]]).astype(np.int32)      # two empty events in between
    emu_ex(w, xy, off2, scheduler=1, steals=steals, debug_bounds=True)
    emu_ex(w, xy, off2, scheduler=1, staging=1, steals=steals, circles=True, peak_mode=1, order="shuffle:5")
    w3 = si.config(3)
    xy3, off3, _ = si.generate(w3, 3)
    big = np.ascontiguousarray(xy3[:off3[3]])
    emu_ex(w3, big, np.array([0, 7, len(big) - 3, len(big)], dtype=np.int32), scheduler=1, steals=steals, threshold=45)
    # clustered grids ignore the option
    emu_ex(w, xy, off, scheduler=1, steals=steals, cluster_size=2)


# ---------------------------------------------------------------- H6 variant: dense selection (HOUGH_OPT_SELECT_MODE)
@pytest.mark.parametrize("cfg,n_ev,kw", [
    (0, 3, dict(select_mode=1, debug_bounds=True)),
    (1, 3, dict(select_mode=1, order="shuffle:4")),
    (2, 2, dict(select_mode=1, debug_bounds=True)),                  # 360 columns: two column groups per hit
    (3, 2, dict(select_mode=2)),                                     # u32, ~800 peaks: the auto mode goes dense
    (1, 3, dict(select_mode=2)),                                     # few peaks: the auto mode keeps the scan
    (0, 3, dict(select_mode=1, theta_wrap=True)),
    (1, 2, dict(select_mode=1, max_peaks=0)),                        # nothing stored: nothing kept, no dense pass
    (1, 2, dict(select_mode=1, peak_mode=1, staging=1, scheduler=1, window=2)),
    (1, 2, dict(select_mode=1, cluster_size=2)),                     # a clustered grid ignores the option
])
def test_dense_selection_under_the_emulator(cfg, n_ev, kw):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    emu_ex(w, xy, off, accum=False, **kw)


def test_dense_selection_with_degenerate_hits_and_a_chunked_event_under_the_emulator():
    w = si.config(0)
    xy, off, _ = si.generate(w, 3)
    bad = np.array([[0, 0], [np.inf, 1], [1e-3, 0], [1e-20, 1e-20], [np.nan, 5], [1e30, 1e30], [3e38, 0]], dtype=np.float32)
    xy2 = np.concatenate([xy[:off[1]], bad, xy[off[1]:]])
    off2 = np.concatenate([[0, 0], off[1:2] + len(bad), off[2:] + len(bad), [off[-1] + len(bad)]]).astype(np.int32)
    emu_ex(w, xy2, off2, accum=False, threshold=5, select_mode=1, grid_clusters=2, debug_bounds=True)   # the exact path of the dense test
    w3 = si.config(3)
    xy3, off3, _ = si.generate(w3, 3)
    big = np.ascontiguousarray(xy3[:off3[3]])                         # one event of ~8000 hits: more than the staging chunk
    g, _ = emu_ex(w3, big, np.array([0, len(big)], dtype=np.int32), accum=False, threshold=40, select_mode=1)
    assert len(big) > g["info"]["CHUNK_HITS"]
