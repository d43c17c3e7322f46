"""Host logic of the library, checked without a GPU: the launch shape and shared-memory layout that
hough_plan_describe() reports (the same planner hough_create uses) must satisfy the invariants the kernel relies on
(DESIGN.md sections 4 and 5)."""
import random

import numpy as np
import pytest

import paper_2607_04067_b200 as hb
import stcf_inputs as si

SMEM_OPTIN = 232448          # B200: 227 KB per CTA with opt-in
SMEM_SM = 233472             # 228 KB per SM, 1 KB reserved per resident CTA
MAGIC_BITS = 0x4B400000


def check_plan(n_theta, n_rho, p):
    C = p["cluster_size"]
    cell = p["acc_bits"] // 8
    assert C in (1, 2, 4, 8, 16)
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
    assert nan_rel >= (n_rho + 1) * p["pitch_bytes"] and nan_rel + p["pitch_bytes"] - 4 <= 0xFFFFFFFF   # largest lane offset: pitch - 4
    # regions follow each other, 16-byte aligned, and fit the CTA's shared memory
    assert p["pbm_off"] == p["region_bytes"]
    assert p["bitmap_words_per_row"] == (n_rho + 31) // 32
    assert p["pbm_bytes"] >= p["cols_per_cta"] * p["bitmap_words_per_row"] * 4
    assert p["pbm_bytes"] >= 8 * n_rho                                   # iterative NMS keeps one 8-byte key per rho row there
    assert 0 < 24 * p["circ_cap"] <= (p["stash_off"] if C > 1 else p["region_bytes"])   # staged circles stay clear of the compaction scratch
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


# ---------------------------------------------------------------- the voting loop's address arithmetic, emulated
CANONICAL_NAN = 0x7FFFFFFF      # what add/mul.f32 produce for a NaN operand (padding columns carry NaN table entries)


def emulate_vote_addresses(p, n_rho, bits):
    """uint32 emulation of hough_kernel.cuh's fast voting path for every lane of the first and last column group:
    rel = min(bits * pitch + lc0, trash0) with lc0 = wbase - MAGIC_BITS * pitch (all mod 2^32), then the ATOMS
    immediates.  Every address must be the lane's own word of row k = bits - MAGIC_BITS when 0 <= k < n_rho, and
    the lane's own word of the trash row (row n_rho) otherwise; nothing may leave the accumulator."""
    M = 0xFFFFFFFF
    pitch, cpl, u16 = p["pitch_bytes"], p["cols_per_lane"], p["acc_bits"] == 16
    bits = np.asarray(bits, dtype=np.uint64)
    k = bits.astype(np.int64) - MAGIC_BITS
    valid = (k >= 0) & (k < n_rho)
    acc_end = (n_rho + 1) * pitch
    imms = sorted({128 * (q // 2) for q in range(0, cpl, 2)} if u16 else {128 * q for q in range(cpl)})
    for g in sorted({0, p["n_groups"] - 1}):
        for lane in range(32):
            wbase = g * (cpl // 2 if u16 else cpl) * 128 + 4 * lane
            lc0 = (wbase - MAGIC_BITS * pitch) & M
            trash0 = n_rho * pitch + wbase
            rel = np.minimum((bits * np.uint64(pitch) + np.uint64(lc0)) & np.uint64(M), np.uint64(trash0)).astype(np.int64)
            assert np.array_equal(rel[valid], k[valid] * pitch + wbase), (g, lane)
            assert np.all(rel[~valid] == trash0), (g, lane, [hex(int(b)) for b in bits[~valid][rel[~valid] != trash0][:4]])
            for imm in imms:
                a = rel + imm
                assert np.all(a + 4 <= acc_end) and np.all(a % 4 == 0)
                assert np.all(a // pitch == np.where(valid, k, n_rho))        # the right row, or the trash row
                assert np.all((a % pitch) // 4 % 32 == lane)                  # lane == bank: conflict-free by construction


def reachable_bits(n_rho, rng, dense):
    """Bit patterns the floor-add can hand to the address arithmetic on the fast path: MAGIC_BITS + floor(t) for
    |t| < 2^17 (tame hits, hough_api.cu tame_bound) and the canonical NaN of a padding column."""
    lim = 1 << 17
    if dense:
        k = np.arange(-lim, lim + 1, dtype=np.int64)
    else:
        k = np.concatenate([np.arange(-300, n_rho + 300), rng.integers(-lim, lim + 1, size=3000), [-lim, lim, -1, 0, n_rho - 1, n_rho]])
    return np.concatenate([(MAGIC_BITS + k).astype(np.uint64), np.array([CANONICAL_NAN], dtype=np.uint64)])


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4, 5])
def test_vote_address_map_of_the_baseline_configs_over_every_reachable_bit_pattern(cfg):
    w = si.config(cfg)
    acc = hb.HOUGH_ACC_U32 if w.acc_dtype == "u32" else hb.HOUGH_ACC_U16
    for C in (0, 2, 4, 8, 16):
        try:
            p = hb.hough_plan_describe(w.n_theta, w.n_rho, acc, cluster_size=C)
        except hb.HoughError:
            continue
        emulate_vote_addresses(p, w.n_rho, reachable_bits(w.n_rho, None, dense=True))


def test_vote_address_map_of_random_grids():
    rng = np.random.default_rng(5)
    pr = random.Random(11)
    done = 0
    for _ in range(400):
        n_theta = pr.choice([1, 2, 31, 33, 64, 65, 180, 193, 360, 384, 500, 720, 1000, 1500, pr.randint(1, 3000)])
        n_rho = pr.choice([1, 2, 31, 32, 33, 128, 256, 257, 512, 1000, pr.randint(1, 2000)])
        acc = pr.choice([hb.HOUGH_ACC_U16, hb.HOUGH_ACC_U32])
        try:
            p = hb.hough_plan_describe(n_theta, n_rho, acc, cluster_size=pr.choice([0, 0, 1, 2, 4, 8, 16]), ctas_per_sm=pr.choice([0, 1]))
        except hb.HoughError:
            continue
        emulate_vote_addresses(p, n_rho, reachable_bits(n_rho, rng, dense=False))
        done += 1
    assert done > 100


def test_only_tame_hits_reach_the_fast_path():
    """The fast path's safety rests on |t| < 2^17 for every (hit, column) it takes.  Emulate the kernel's tame test and
    S2 in numpy fp32 for adversarial hits at and around the bound, for every baseline grid: a hit that passes the test
    has |t| < 2^17 at every column and no subnormal product; NaN / inf / huge / subnormal (u, v) never pass."""
    f32 = np.float32
    for cfg in range(6):
        w = si.config(cfg)
        c, s = si.trig_table(w.n_theta)
        tab = np.concatenate([np.abs(c), np.abs(s)])
        tmax, tmin_nz = float(tab.max()), float(tab[tab > 0].min())
        bound, ftz_min = hb.hough_debug_tame_bounds(w.n_rho, w.rho_max, tmax, tmin_nz)
        inv = f32(float(w.n_rho) / (2.0 * float(f32(w.rho_max))))
        rng = np.random.default_rng(cfg)
        mags = np.concatenate([bound * np.array([1e-6, 0.1, 0.5, 0.9, 0.99, 0.999999, 1.0, 1.000001, 1.01, 2.0, 1e3]),
                               [0.0, ftz_min * 0.5, ftz_min, ftz_min * 2, 1e-45, 1e-38, 3e38, np.inf, np.nan]])
        phi = rng.uniform(0, 2 * np.pi, size=64)
        U = np.concatenate([np.outer(mags, np.cos(phi)).ravel(), mags, np.zeros_like(mags), -mags]).astype(f32)
        V = np.concatenate([np.outer(mags, np.sin(phi)).ravel(), np.zeros_like(mags), mags, mags]).astype(f32)
        with np.errstate(all="ignore"):
            au, av = np.abs(U), np.abs(V)
            tame = ((au + av).astype(f32) <= f32(bound)) & ((au >= f32(ftz_min)) | (au == 0)) & ((av >= f32(ftz_min)) | (av == 0))
            assert not tame[~np.isfinite(U) | ~np.isfinite(V)].any()
            assert tame.any() and (~tame).any()
            Ut, Vt = U[tame][:, None], V[tame][:, None]
            p1, p2 = (Ut * c[None, :]).astype(f32), (Vt * s[None, :]).astype(f32)
            t = (((p1 + p2).astype(f32) + f32(w.rho_max)).astype(f32) * inv).astype(f32)
            assert np.all(np.abs(t) < 2.0 ** 17), (cfg, float(np.abs(t).max()))
            tiny = f32(2.0 ** -126)
            assert np.all((np.abs(p1) >= tiny) | (p1 == 0) & ((Ut == 0) | (c[None, :] == 0)))
            assert np.all((np.abs(p2) >= tiny) | (p2 == 0) & ((Vt == 0) | (s[None, :] == 0)))


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
    for C in (1, 2, 4, 8, 16):
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


def test_the_papers_own_grid_takes_a_16_cta_cluster():
    # 1000 x 1000 needs 2 MB of u16 cells: beyond an 8-CTA cluster, 63 columns per CTA of a 16-CTA one
    # (SURVEY.md 8(f) NEXT-3); 4 MB of u32 cells fit nowhere
    p = hb.hough_plan_describe(1000, 1000, hb.HOUGH_ACC_U16)
    assert (p["cluster_size"], p["cols_per_cta"], p["threads"]) == (16, 63, 1024)
    check_plan(1000, 1000, p)
    emulate_vote_addresses(p, 1000, reachable_bits(1000, None, dense=True))
    with pytest.raises(hb.HoughError):
        hb.hough_plan_describe(1000, 1000, hb.HOUGH_ACC_U32)
    # 16 is only taken when nothing smaller fits
    assert hb.hough_plan_describe(360, 512, hb.HOUGH_ACC_U16)["cluster_size"] == 2


def test_bad_arguments_are_rejected():
    for args in ((0, 10), (10, 0), (70000, 10), (10, 70000)):
        with pytest.raises(hb.HoughError):
            hb.hough_plan_describe(*args)
    with pytest.raises(hb.HoughError):
        hb.hough_plan_describe(10, 10, 7)
    with pytest.raises(hb.HoughError):
        hb.hough_plan_describe(10, 10, hb.HOUGH_ACC_U16, cluster_size=3)
