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
    emu_only = {k: args.pop(k) for k in ("cluster_size", "ctas_per_sm", "vote_path", "grid_clusters", "debug_bounds") if k in args}
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
