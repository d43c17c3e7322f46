"""Host logic of the library, checked without a GPU: the launch shape and shared-memory layout that
hough_plan_describe() reports (the same planner hough_create uses) must satisfy the invariants the kernel relies on
(DESIGN.md sections 4 and 5)."""
import random

import pytest

import paper_2607_04067_b200 as hb
import stcf_inputs as si

SMEM_OPTIN = 232448          # B200: 227 KB per CTA with opt-in
SMEM_SM = 233472             # 228 KB per SM, 1 KB reserved per resident CTA
MAGIC_BITS = 0x4B400000


def check_plan(n_theta, n_rho, p):
    C = p["cluster_size"]
    cell = p["acc_bits"] // 8
    assert C in (1, 2, 4, 8)
    assert p["cols_per_cta"] * C >= n_theta and p["cols_per_cta"] * (C - 1) < n_theta
    # vote mapping: every warp owns one group of 32 * CPL columns, all groups together cover the CTA's columns
    padded = 32 * p["cols_per_lane"] * p["n_groups"]
    assert padded >= p["cols_per_cta"]
    assert p["threads"] == 32 * p["n_groups"] * p["n_stripes"] and 32 <= p["threads"] <= 1024
    # rho-major rows: one 128-byte line per 32 lanes, so lane = bank whatever the rho bin is
    assert p["pitch_bytes"] == padded * cell and p["pitch_bytes"] % 128 == 0 and p["pitch_bytes"] <= 8192
    assert p["region_bytes"] >= (n_rho + 1) * p["pitch_bytes"]          # + the trash row
    # a bin of magnitude < 2^17 (tame hits) times the pitch never wraps a 32-bit offset
    assert (1 << 17) * p["pitch_bytes"] < (1 << 31)
    # padding columns carry NaN table entries: their offset must fall beyond the accumulator for every word of a row
    nan_rel = ((0x7FFFFFFF - MAGIC_BITS) * p["pitch_bytes"]) & 0xFFFFFFFF
    assert nan_rel >= (n_rho + 1) * p["pitch_bytes"] and nan_rel + p["pitch_bytes"] <= 0xFFFFFFFF
    # regions follow each other, 16-byte aligned, and fit the CTA's shared memory
    assert p["pbm_off"] == p["region_bytes"]
    assert p["bitmap_words_per_row"] == (n_rho + 31) // 32
    assert p["pbm_bytes"] >= p["cols_per_cta"] * p["bitmap_words_per_row"] * 4
    assert p["hb_off"] == p["pbm_off"] + p["pbm_bytes"]
    assert p["misc_off"] == p["hb_off"] + 8 * p["chunk_hits"]
    assert p["smem_bytes"] >= p["misc_off"] + 256 and p["smem_bytes"] <= SMEM_OPTIN
    for k in ("region_bytes", "pbm_off", "hb_off", "misc_off", "w8_off", "w8_pitch", "mcf_off", "msf_off", "colq_off",
              "stash_off", "cnt_off", "gcnt_off"):
        assert p[k] % 16 == 0, k
    assert 128 <= p["chunk_hits"] <= 4096 and p["chunk_hits"] % 2 == 0
    # selection data reuses the (dead) accumulator region: in order, no overlap, inside the region
    assert p["w8_pitch"] >= n_rho + 1
    assert p["mcf_off"] >= p["w8_off"] + ((n_theta + 7) // 8) * p["w8_pitch"]
    assert p["msf_off"] >= p["mcf_off"] + 4 * (n_theta + 8)
    assert p["colq_off"] >= p["msf_off"] + 4 * (n_theta + 8)
    assert p["stash_off"] >= p["colq_off"] + 4 * n_theta
    assert p["stash_off"] <= p["cnt_off"] <= p["gcnt_off"] <= p["region_bytes"]
    if C > 1:
        nwarps = p["threads"] // 32
        assert p["cnt_off"] >= p["stash_off"] + 32 * nwarps * 4
        assert p["gcnt_off"] >= p["cnt_off"] + 32 * 4
        assert p["region_bytes"] >= p["gcnt_off"] + (32 * C + 1) * 4
    # the division-free index arithmetic of the kernel is exact over its whole domain
    for w in range(32):
        assert (w * p["rcp_groups"]) >> 16 == w // p["n_groups"]
    for m in range(p["chunk_hits"] + 1):
        assert (m * p["rcp_2s"]) >> 20 == m // (2 * p["n_stripes"])
        assert m * p["rcp_2s"] < (1 << 32)


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4, 5])
def test_plans_of_the_baseline_configs(cfg):
    w = si.config(cfg)
    acc = hb.HOUGH_ACC_U32 if w.acc_dtype == "u32" else hb.HOUGH_ACC_U16
    p = hb.hough_plan_describe(w.n_theta, w.n_rho, acc)
    check_plan(w.n_theta, w.n_rho, p)
    expect = {0: (1, 512), 1: (1, 512), 2: (1, 1024), 3: (1, 1024), 4: (1, 512), 5: (2, 1024)}[cfg]
    assert (p["cluster_size"], p["threads"]) == expect
    if p["threads"] == 512:          # two CTAs of this plan are resident per SM
        assert 2 * (p["smem_bytes"] + 1024) <= SMEM_SM
    # a nominal event (<= 1100 hits) is staged in one piece for the headline configs
    if cfg in (1, 4):
        assert p["chunk_hits"] >= 1100


def test_forced_cluster_sizes_and_one_cta_per_sm():
    for C in (1, 2, 4, 8):
        p = hb.hough_plan_describe(360, 256, hb.HOUGH_ACC_U16, cluster_size=C)
        assert p["cluster_size"] == C
        check_plan(360, 256, p)
    p = hb.hough_plan_describe(180, 256, hb.HOUGH_ACC_U16, ctas_per_sm=1)
    assert p["threads"] == 1024
    check_plan(180, 256, p)


def test_random_grids_either_fit_with_all_invariants_or_are_refused():
    rng = random.Random(7)
    fitted = refused = 0
    for _ in range(300):
        n_theta = rng.choice([1, 2, 31, 32, 33, 64, 65, 180, 192, 193, 360, 384, 500, 720, 1000, 1500, rng.randint(1, 3000)])
        n_rho = rng.choice([1, 2, 31, 32, 33, 128, 256, 257, 512, 1000, rng.randint(1, 2000)])
        acc = rng.choice([hb.HOUGH_ACC_U16, hb.HOUGH_ACC_U32])
        try:
            p = hb.hough_plan_describe(n_theta, n_rho, acc)
        except hb.HoughError:
            refused += 1
            continue
        check_plan(n_theta, n_rho, p)
        fitted += 1
    assert fitted > 100 and refused > 0


def test_the_papers_own_grid_is_refused_for_now():
    # 1000 x 1000 needs 2 MB of u16 cells: beyond an 8-CTA cluster
    with pytest.raises(hb.HoughError):
        hb.hough_plan_describe(1000, 1000, hb.HOUGH_ACC_U16)


def test_bad_arguments_are_rejected():
    for args in ((0, 10), (10, 0), (70000, 10), (10, 70000)):
        with pytest.raises(hb.HoughError):
            hb.hough_plan_describe(*args)
    with pytest.raises(hb.HoughError):
        hb.hough_plan_describe(10, 10, 7)
    with pytest.raises(hb.HoughError):
        hb.hough_plan_describe(10, 10, hb.HOUGH_ACC_U16, cluster_size=3)
