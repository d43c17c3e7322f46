"""-m "not gpu": the scenarios of the `-m gpu` parity tests (tests/test_parity_gpu.py, tests/test_parity_next_gpu.py), run
through the SIMT emulator of tests/simt_emu with the bounds-checked flavour of the kernel source.  The GPU tests'
own functions are called with their `gpu_run` / `gpu_ex` helper swapped for an emulator-backed one, so the inputs,
options and assertions are exactly the ones the GPU will see.  This checks the kernel's logic and the design of those
tests on a box without a GPU; it is not the parity gate (see tests/simt_emu/__init__.py)."""
import numpy as np
import pytest

import oracle
import paper_2607_04067_b200 as hb
import stcf_inputs as si
import tests.test_parity_next_gpu as tn
import tests.test_parity_gpu as tp
from tests import simt_emu


def emu_gpu_run(_hb, xy, off, n_theta, n_rho, rho_max, threshold, window, table, max_peaks=64, acc_dtype="u16", accum=True,
                conformal_scale=1, cluster_size=0, ctas_per_sm=0, vote_path=0, stream=None):
    table = si.trig_table(n_theta) if table is None else table
    g = simt_emu.run(xy, off, n_theta, n_rho, rho_max, threshold, window, table, max_peaks=max_peaks, acc_dtype=acc_dtype,
                     accum=accum, conformal_scale=conformal_scale, cluster_size=cluster_size, ctas_per_sm=ctas_per_sm,
                     vote_path=vote_path, debug_bounds=True)
    assert not np.any(g["counts"][:, 0] == -2), "debug-bounds sentinel: phases %s" % g["counts"][g["counts"][:, 0] == -2, 1]
    return g


def emu_gpu_ex(_hb, w, xy, off, accum=True, circles=False, cluster_size=0, rho_max=None, **kw):
    table = si.trig_table(w.n_theta)
    base = dict(max_peaks=w.max_peaks, acc_dtype=w.acc_dtype, threshold=w.threshold, window=w.window, conformal_scale=1)
    base.update({k: kw.pop(k) for k in list(kw) if k in base})
    opts = {k: kw.pop(k) for k in list(kw) if k in tn.OPTS}
    emu_only = {k: kw.pop(k) for k in list(kw) if k in tn.GPU_ONLY}
    assert not kw, kw
    rho_max = w.rho_max if rho_max is None else rho_max
    g = simt_emu.run(xy, off, w.n_theta, w.n_rho, rho_max, base["threshold"], base["window"], table, max_peaks=base["max_peaks"],
                     acc_dtype=base["acc_dtype"], accum=accum, conformal_scale=base["conformal_scale"], circles=circles,
                     cluster_size=cluster_size, debug_bounds=True, **opts, **emu_only)
    assert not np.any(g["counts"][:, 0] == -2), "debug-bounds sentinel"
    o, oc = oracle.run_ex(xy, off, w.n_theta, w.n_rho, rho_max, base["threshold"], base["window"], table[0], table[1],
                          max_peaks=base["max_peaks"], conformal_scale=base["conformal_scale"], acc_u16=(base["acc_dtype"] != "u32"),
                          want_accum=accum, n_threads=4, want_circles=circles, **opts)
    tp.compare(g, o, off, base["max_peaks"], accum=accum, tag=w.name)
    if circles:
        for e in range(len(off) - 1):
            ns = min(int(o.counts[e, 0]), base["max_peaks"])
            assert g["circles"][e, :ns].tobytes() == oc[e, :ns].tobytes(), "circles of event %d" % e
    return g, o, oc


@pytest.fixture()
def emulated(monkeypatch):
    monkeypatch.setattr(tp, "gpu_run", emu_gpu_run)
    monkeypatch.setattr(tn, "gpu_ex", emu_gpu_ex)
    return hb


PARITY = [
    ("test_forced_cluster_of_eight_matches_oracle", ()),
    ("test_cluster_grid_360x512_u32_plans_eight_ctas", ()),
    ("test_cluster_with_degenerate_hits_takes_the_slow_path", (2,)),
    ("test_cluster_with_degenerate_hits_takes_the_slow_path", (8,)),
    ("test_cluster_with_an_event_larger_than_the_staging_chunk", (2, "u16")),
    ("test_cluster_with_an_event_larger_than_the_staging_chunk", (4, "u32")),
    ("test_cluster_with_max_peaks_truncation", (0,)),
    ("test_cluster_with_max_peaks_truncation", (3,)),
    ("test_cluster_with_windows", (2, 2)),
    ("test_cluster_with_windows", (8, 3)),
    ("test_cluster_selection_runs_a_second_round", ()),
    ("test_event_larger_than_the_staging_chunk", ()),
    ("test_one_cta_per_sm_and_slow_vote_path", ()),
    ("test_tiny_and_odd_grids", ()),
    ("test_empty_and_ragged_events", ()),
    ("test_degenerate_hits_take_the_exact_slow_path", ()),
    ("test_u16_overflow_event_is_refused", ()),
    ("test_conformal_scale_2", ()),
    ("test_default_trig_table_equals_harness_table", ()),
    ("test_p1_closed_form_on_gpu", ()),
    ("test_power_of_two_row_pitch_grid", ()),
] + [("test_every_kernel_instantiation", inst) for inst in tp.INSTANTIATIONS]

NEXT = [
    ("test_n1_circles_match_the_oracle_bit_for_bit", (2, 3)),
    ("test_n1_circles_match_the_oracle_bit_for_bit", (3, 2)),
    ("test_n1_closed_form_worked_example_scale_2_and_b_field", ()),
    ("test_n1_on_a_cluster_grid_and_with_empty_and_refused_events", ()),
    ("test_n2_relative_threshold_and_iterative_nms", (2, 3, 400, 1)),
    ("test_n2_relative_threshold_and_iterative_nms", (3, 2, 700, 3)),
    ("test_n2_relative_threshold_and_iterative_nms", (1, 6, 0, 0)),
    ("test_n2_relative_threshold_and_iterative_nms", (1, 6, 1000, 5)),
    ("test_n4a_theta_wrap", (8, 1)),
    ("test_n4a_theta_wrap", (0, 3)),
    ("test_n4b_distance_filter", (1, 6, 4, 20.0)),
    ("test_n4b_distance_filter", (3, 2, 0, 0.5)),
    ("test_n4b_more_stored_peaks_than_staged_circles", ()),
    ("test_n2_with_theta_wrap_and_on_cluster_grids", ()),
    ("test_h0_bulk_copy_staging", (0, 16, 0)),
    ("test_h0_bulk_copy_staging", (1, 8, 4)),
    ("test_h0_bulk_copy_staging", (5, 2, 0)),
    ("test_work_stealing_scheduler", (0, 16, 0)),
    ("test_work_stealing_scheduler", (1, 12, 1)),
]


@pytest.mark.parametrize("name,args", PARITY, ids=["%s%s" % (n[5:], list(a)) for n, a in PARITY])
def test_parity_scenario(emulated, name, args):
    getattr(tp, name)(emulated, *args)


@pytest.mark.parametrize("name,args", NEXT, ids=["%s%s" % (n[5:], list(a)) for n, a in NEXT])
def test_next_scenario(emulated, name, args):
    getattr(tn, name)(emulated, *args)
