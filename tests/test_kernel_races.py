"""Race check of the kernel without a GPU (the stand-in for `compute-sanitizer --tool racecheck` while GPU access is
closed).  The kernel source runs under the SIMT emulator built with the compiler's
-fsanitize=thread instrumentation and the emulator's OWN runtime (tests/simt_emu/simt_shim.h): every memory access of
the kernel is checked against the last write, the last atomics and the reads since of the same byte -- shared memory of
every CTA of the cluster (DSMEM included) and the global output buffers.  Two accesses of different CUDA threads, at
least one a write, not both atomic, are a race unless a barrier both threads share lies between them (__syncwarp,
__syncthreads*, cluster.sync; for cp.async.bulk / launch-control writes: the mbarrier phase the reader waited for).
Warp shuffles and votes order nothing; threads of different clusters are never ordered.  The same shadow state gives
an initcheck: a read or atomic of a byte nothing has written yet is reported too.  The mutation tests prove the
detector detects: the same scenarios with one barrier removed, or one atomic made a plain store, must be reported at
the lines involved."""
import os
import re
import shutil
import subprocess
import sys
import tempfile

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)
sys.path.insert(0, os.path.dirname(HERE))

import simt_emu  # noqa: E402
import stcf_inputs as si  # noqa: E402


@pytest.fixture(scope="module")
def race_exe():
    return simt_emu.build(race=True)


def race_run(cfg, nev, exe=None, n_theta=None, n_rho=None, **kw):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, nev)
    nt, nr = n_theta or w.n_theta, n_rho or w.n_rho
    return simt_emu.run(xy, off, nt, nr, w.rho_max, w.threshold, w.window, si.trig_table(nt), max_peaks=kw.pop("max_peaks", w.max_peaks),
                        acc_dtype=kw.pop("acc_dtype", w.acc_dtype), accum=False, race=True, exe=exe, timeout=1500, **kw)


# every instantiation family and every optional path, several events per CTA (grid_clusters = 1: the event loop's
# re-use of shared memory is part of what is checked), three scheduling orders
SCENARIOS = {
    "cfg0 u16, 3 events through one CTA": dict(cfg=0, nev=3, grid_clusters=1),
    "cfg0 u32": dict(cfg=0, nev=2, grid_clusters=1, acc_dtype="u32"),
    "cfg1 (two chunks per event), reverse order": dict(cfg=1, nev=2, grid_clusters=1, order="reverse"),
    "cfg1, shuffled order": dict(cfg=1, nev=2, grid_clusters=1, order="shuffle:7"),
    "cfg1, peak list saturated": dict(cfg=1, nev=2, grid_clusters=1, max_peaks=4),
    "cfg2 (1024 threads)": dict(cfg=2, nev=2, grid_clusters=1),
    "exact slow path, cluster of 2": dict(cfg=1, nev=2, grid_clusters=1, cluster_size=2, vote_path=1),
    "cluster of 2, u32": dict(cfg=0, nev=2, grid_clusters=1, cluster_size=2, acc_dtype="u32"),
    "cluster of 4, shuffled": dict(cfg=1, nev=2, grid_clusters=1, cluster_size=4, order="shuffle:1"),
    "cluster of 8": dict(cfg=0, nev=2, grid_clusters=1, cluster_size=8),
    "N2 iterative NMS": dict(cfg=1, nev=2, grid_clusters=1, peak_mode=1, order="shuffle:5"),
    "N2 iterative NMS, cluster of 4": dict(cfg=0, nev=2, grid_clusters=1, cluster_size=4, peak_mode=1),
    "N4a wrap + N4b distance filter + N1 circles, cluster of 2, bulk staging": dict(
        cfg=1, nev=3, grid_clusters=1, cluster_size=2, peak_mode=1, theta_wrap=True, keep_mode=1, keep_tol=5.0, staging=1, circles=True),
    "bulk staging + work stealing": dict(cfg=1, nev=5, grid_clusters=2, staging=1, scheduler=1),
    "dense selection, 3 events through one CTA": dict(cfg=3, nev=3, grid_clusters=1, select_mode=1),
    "dense selection, two column groups, shuffled": dict(cfg=2, nev=2, grid_clusters=1, select_mode=1, order="shuffle:9"),
    "work stealing, cluster of 2": dict(cfg=0, nev=3, cluster_size=2, scheduler=1),
}


@pytest.mark.parametrize("name", list(SCENARIOS))
def test_no_data_race(race_exe, name):
    race_run(**SCENARIOS[name])          # raises simt_emu.RaceReport: both accesses with function, file and line


def test_no_data_race_in_the_16_cta_cluster_of_the_papers_grid(race_exe):
    """PAPER.md:73's 1000 x 1000 grid: 16 CTAs of 1024 threads, every DSMEM exchange of the cluster path."""
    r = race_run(1, 1, n_theta=1000, n_rho=1000, acc_dtype="u16")
    assert r["info"]["CLUSTER_SIZE"] == 16


# ---- the detector detects: mutants of the kernel source.  (old text, new text), the scenario, and a line of the kernel
# that must appear in a report
MUTANTS = {
    "the barrier after the voting loop removed": (
        [("            __syncthreads();\n        }\n        if (n == 0) __syncthreads();         // no staging barrier ran",
          "        }\n        if (n == 0) __syncthreads();         // no staging barrier ran")],
        dict(cfg=0, nev=1), "atomicAdd"),
    "cluster barrier (A) between the votes and the remote halo reads of H4 removed": (
        [("        if (CL) cg::this_cluster().sync();   // (A) every CTA's columns are complete", "        // (A) removed")],
        dict(cfg=1, nev=1, cluster_size=8), "atomicAdd"),      # 24 columns per CTA: above-threshold cells on CTA borders
    "cluster barrier (E) before the next round's counts are rewritten removed": (
        [("                cg::this_cluster().sync();   // (E) remote reads of cnt done", "                // (E) removed")],
        dict(cfg=1, nev=2, grid_clusters=1, cluster_size=2), "cnt"),
    "the column marks of overlapping peak windows as plain stores": (
        [("            for (int j = jlo; j <= jhi; ++j)\n                if (HB_CHK(j >= 0 && j < p.n_theta, HB_H6_SETUP)) atomicOr(&colq[j], 1);",
          "            for (int j = jlo; j <= jhi; ++j)\n                if (HB_CHK(j >= 0 && j < p.n_theta, HB_H6_SETUP)) colq[j] = 1;")],
        dict(cfg=0, nev=2, grid_clusters=1), "colq[j] = 1"),
    "block_exscan called back to back without the __syncwarp": (
        [("    __syncwarp();                        // a previous call's reads of wsum[warp]", "    // removed: a previous call's reads of wsum[warp]")],
        dict(cfg=1, nev=1), "wsum[warp]"),
    "initcheck: the vector-list counter not reset before H4 counts with it": (
        [("if (tid == 0) { misc[42] = 0; misc[33] = 1; }", "if (tid == 0) { misc[33] = 1; }")],
        dict(cfg=0, nev=1), "misc[42]"),
    "bulk-copy staging: the hits read without waiting for the mbarrier": (
        [("                    bool done = false;\n                    for (int spin = 0; spin < (1 << 24) && !done; ++spin) done = mbar_try_wait(bar_s, bar_phase);",
          "                    bool done = true;")],
        dict(cfg=1, nev=1, staging=1), "hb["),
}


@pytest.fixture(scope="module")
def mutant_exes():
    """All mutants compiled at once (one g++ each, in parallel)."""
    from concurrent.futures import ThreadPoolExecutor
    d = tempfile.mkdtemp(prefix="hough_mut_")
    names = list(MUTANTS)
    try:
        with ThreadPoolExecutor(len(names)) as ex:
            exes = list(ex.map(lambda i: simt_emu.build_mutant(os.path.join(d, "emu_mut%d" % i), MUTANTS[names[i]][0]), range(len(names))))
        yield dict(zip(names, exes))
    finally:
        shutil.rmtree(d, ignore_errors=True)


@pytest.mark.parametrize("name", list(MUTANTS))
def test_mutant_is_reported(mutant_exes, name):
    _, scenario, needle = MUTANTS[name]
    exe = mutant_exes[name]
    with pytest.raises(simt_emu.RaceReport) as info:
        race_run(exe=exe, **scenario)
    src = open(exe + ".cuh").read().splitlines()
    lines = []
    for r in info.value.reports:
        for m in re.finditer(r"emu_mut\d+\.cuh:(\d+)", r["now"] + " " + r["earlier"]):
            lines.append(src[int(m.group(1)) - 1])
    assert any(needle in l for l in lines), (needle, lines[:6], str(info.value)[:1500])


def test_synccheck_a_barrier_reached_from_two_call_sites_is_refused():
    """The emulator's synccheck: all threads of a barrier generation must come from the same barrier call of the source."""
    d = tempfile.mkdtemp(prefix="hough_mut_")
    try:
        exe = simt_emu.build_mutant(os.path.join(d, "emu_sync"), [
            ("            __syncthreads();   // D / lists are dead: the region may be zeroed for the next event",
             "            if (tid & 32) __syncthreads();\n            else __syncthreads();")], race=False)
        w = si.config(0)
        xy, off, _ = si.generate(w, 1)
        with pytest.raises(RuntimeError, match="divergent barrier"):
            simt_emu.run(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, si.trig_table(w.n_theta), max_peaks=w.max_peaks,
                         acc_dtype=w.acc_dtype, accum=False, exe=exe)
    finally:
        shutil.rmtree(d, ignore_errors=True)
