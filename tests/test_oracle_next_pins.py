"""-m "not gpu": pins of oracle/hough_oracle_next.cpp (the NEXT rows N1, N2, N4a, N4b of SURVEY.md 8(f)) against what
the paper and the mathematics fix: the hand-worked rows of tests/golden/w1_next.txt, the closed form of a circle
through the origin (Eq. (1)/(2)), pT = 0.3 B R, exact rescaling, independent numpy
restatements and invariants.  Also pins S3 of the ORIGINAL oracle on crafted accumulators (oracle.find_peaks)."""
import os

import numpy as np
import pytest

import oracle
import stcf_inputs as si
from tests import np_model as npm

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "w1_next.txt")
W1_XY = np.array([[1, 0], [0, 1], [.5, .5], [-1, 0], [0, 0], [4, 0]], dtype=np.float32)
W1_OFF = np.array([0, 6], dtype=np.int32)
W1_A = np.array([[0, 0, 1, 0, 2, 0, 2, 0], [0, 0, 1, 0, 1, 2, 1, 0], [0, 0, 0, 0, 3, 0, 2, 0], [0, 0, 1, 1, 1, 2, 0, 0]], dtype=np.uint32)


def gold_sections():
    sec, cur = {}, None
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line[0].isalpha():
            cur = line
            sec[cur] = []
        else:
            sec[cur].append([float(t) for t in line.split()])
    return sec


def w1(**kw):
    t = si.trig_table(4)
    args = dict(threshold=2, window=0, max_peaks=8)
    args.update(kw)
    thr, w = args.pop("threshold"), args.pop("window")
    return oracle.run_ex(W1_XY, W1_OFF, 4, 8, 2.0, thr, w, t[0], t[1], **args)


# ---------------------------------------------------------------- golden rows
def test_w1_circles_match_the_hand_worked_rows():
    rows = gold_sections()["circles thr=2 w=0"]
    r, c = w1(want_circles=True)
    assert r.counts[0, 0] == 3
    for q, (j, k, xc, yc, rc, pt, phi0_over_pi, ch, nh) in enumerate(rows):
        assert r.peaks[0, q, :2].tolist() == [j, k]
        assert c[0, q]["x_c"] == pytest.approx(xc, rel=1e-6, abs=1e-22) and c[0, q]["y_c"] == pytest.approx(yc, rel=1e-12)
        assert c[0, q]["r_c"] == pytest.approx(rc, rel=1e-12) and c[0, q]["pt"] == pytest.approx(pt, rel=1e-12)
        assert c[0, q]["phi0"] == pytest.approx(phi0_over_pi * np.pi, abs=1e-12)
        assert (c[0, q]["charge"], c[0, q]["n_hits"]) == (ch, nh)


def test_w1_nms_sequences_match_the_hand_worked_rows():
    g = gold_sections()
    for key, (pm, rad) in (("nms thr=2 permille=500 radius=1", (500, 1)), ("nms thr=2 permille=1000 radius=1", (1000, 1)),
                           ("nms thr=2 permille=500 radius=2", (500, 2))):
        n, p = oracle.find_peaks_ex(W1_A, 2, peak_mode=1, rel_permille=pm, nms_radius=rad)
        assert n == len(g[key]) and p.tolist() == [[int(v) for v in row] for row in g[key]], key
        r, _ = w1(peak_mode=1, rel_permille=pm, nms_radius=rad, want_accum=True)      # the same through a whole event
        assert np.array_equal(r.accum[0], W1_A) and r.counts[0, 0] == n and np.array_equal(r.peaks[0, :n], p)


def test_w1_wrap_and_distance_keep_masks_match_the_hand_worked_rows():
    g = gold_sections()
    for wrap in (0, 1):
        r, _ = w1(window=1, max_peaks=1, theta_wrap=bool(wrap))
        assert r.peaks[0, 0].tolist() == [0, 4, 2]
        assert r.keep.tolist() == [int(v) for v in g["keep thr=2 w=1 max_peaks=1 wrap=%d" % wrap][0]]
    for tol in ("0.1", "0.3", "0.5"):
        r, _ = w1(threshold=3, keep_mode=1, keep_tol=float(tol))
        assert r.keep.tolist() == [int(v) for v in g["keep_distance thr=3 tol=" + tol][0]], tol
        assert r.counts[0].tolist() == [1, int(sum(g["keep_distance thr=3 tol=" + tol][0]))]


def test_seam_example_of_the_wrapped_3x3_rule():
    A = np.zeros((3, 4), dtype=np.uint32)
    A[0, 1] = A[2, 2] = 5
    assert oracle.find_peaks_ex(A, 1)[1].tolist() == [[0, 1, 5], [2, 2, 5]]
    assert oracle.find_peaks_ex(A, 1, theta_wrap=True)[1].tolist() == [[2, 2, 5]]
    A[0, 1] = 6
    assert oracle.find_peaks_ex(A, 1, theta_wrap=True)[1].tolist() == [[0, 1, 6]]


# ---------------------------------------------------------------- S3 of the original oracle on crafted accumulators
def test_original_s3_plateau_border_and_diagonal_rules():
    A = np.zeros((5, 6), dtype=np.uint32)
    A[2, 2] = A[2, 3] = 7          # horizontal plateau -> the raster-first cell only (reading Q8)
    A[0, 0] = 5                    # corner: outside counts as 0
    A[4, 5] = 5
    A[0, 5] = 4; A[1, 4] = 4       # diagonal tie: (0,5) precedes (1,4)
    n, p = oracle.find_peaks(A, 4)
    assert n == 4 and p.tolist() == [[0, 0, 5], [0, 5, 4], [2, 2, 7], [4, 5, 5]]
    n, p = oracle.find_peaks(A, 4, max_peaks=2)            # S4: truncation keeps the raster-first, counts all
    assert n == 4 and p.tolist() == [[0, 0, 5], [0, 5, 4]]
    assert oracle.find_peaks(W1_A, 2)[1].tolist() == [[0, 4, 2], [0, 6, 2], [2, 4, 3]]
    assert oracle.find_peaks(A, 8)[0] == 0


def test_restated_steps_equal_the_pinned_ones_when_every_option_is_off():
    rng = np.random.default_rng(3)
    for _ in range(20):
        A = rng.poisson(1.2, size=(rng.integers(1, 30), rng.integers(1, 30))).astype(np.uint32)
        a, b = oracle.find_peaks(A, 2), oracle.find_peaks_ex(A, 2)
        assert a[0] == b[0] and np.array_equal(a[1], b[1])
    for cfg in (0, 1):
        w = si.config(cfg)
        xy, off, _ = si.generate(w, 3)
        t = si.trig_table(w.n_theta)
        r0 = oracle.run(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], max_peaks=w.max_peaks, want_accum=True)
        r1, _ = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], max_peaks=w.max_peaks, want_accum=True)
        for f in ("keep", "peaks", "counts", "kept_xy", "kept_idx", "accum"):
            assert np.array_equal(getattr(r0, f), getattr(r1, f)), f


# ---------------------------------------------------------------- N1: closed form of a circle through the origin
def p1_hits(q, mirrored=False, nt=180, jstar=40, kstar=70):
    inv = 21376.0
    R = 1.0 / (2.0 * ((kstar + 0.5) / inv - float(si.RHO_MAX)))
    r = 200.0 + np.arange(48) * 600.0 / 47.0
    phi_c = jstar * np.pi / nt + (np.pi if mirrored else 0.0)
    phi = phi_c - q * np.arccos(r / (2 * R))                 # the input recipe's outgoing branch
    return np.stack([r * np.cos(phi), r * np.sin(phi)], axis=1).astype(np.float32), R, phi_c


@pytest.mark.parametrize("q", [1, -1])
@pytest.mark.parametrize("mirrored", [False, True])
def test_n1_closed_form_radius_centre_direction_charge_and_phi0(q, mirrored):
    xy, R, phi_c = p1_hits(q, mirrored)
    t = si.trig_table(180)
    r, c = oracle.run_ex(xy, np.array([0, 48], dtype=np.int32), 180, 128, si.RHO_MAX, 20, 1, t[0], t[1], want_circles=True, b_field=1.0)
    stored = r.peaks[0, :r.counts[0, 0]].tolist()
    want = [40, 57 if mirrored else 70, 48]
    assert want in stored
    ci = c[0, stored.index(want)]
    half_bin = 0.5 / 21376.0                                  # in rho; dR = R^2 * 2 * drho
    assert abs(ci["r_c"] - R) <= 2 * R * R * half_bin and ci["r_c"] == pytest.approx(1644.31, abs=0.01)
    assert ci["pt"] == pytest.approx(0.3 * 1.0 * R * 1e-3, rel=1e-6) and ci["pt"] == pytest.approx(0.4933, abs=1e-4)
    assert np.hypot(ci["x_c"], ci["y_c"]) == pytest.approx(ci["r_c"], rel=1e-6)     # the circle passes through the origin
    assert np.arctan2(ci["y_c"], ci["x_c"]) % (2 * np.pi) == pytest.approx(phi_c % (2 * np.pi), abs=1e-6)
    assert ci["charge"] == q and ci["n_hits"] == 48
    assert ci["phi0"] == pytest.approx((phi_c - q * np.pi / 2) % (2 * np.pi), abs=1e-9)
    # every hit lies on the candidate circle to within half a rho bin
    d = np.hypot(xy[:, 0].astype(np.float64) - ci["x_c"], xy[:, 1].astype(np.float64) - ci["y_c"])
    assert np.abs(d - ci["r_c"]).max() < 2 * R * R * half_bin * 1.05 + 1e-3


def test_n1_b_field_scales_pt_and_scale_2_is_bit_identical():
    xy, R, _ = p1_hits(1)
    off = np.array([0, 48], dtype=np.int32)
    t = si.trig_table(180)
    _, c1 = oracle.run_ex(xy, off, 180, 128, si.RHO_MAX, 20, 1, t[0], t[1], want_circles=True, b_field=1.0)
    _, c2 = oracle.run_ex(xy, off, 180, 128, si.RHO_MAX, 20, 1, t[0], t[1], want_circles=True, b_field=0.5)
    assert np.array_equal(c2["pt"][0, :1] * 2, c1["pt"][0, :1]) and np.array_equal(c1["r_c"], c2["r_c"])
    # Eq. (2) as printed goes with u = 2x/(x^2+y^2): (scale 2, 2 rho_max) is the same circle, bit for bit (reading Q1)
    w = si.config(0)
    xy, off, _ = si.generate(w, 4)
    ra, ca = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], want_circles=True)
    rb, cb = oracle.run_ex(xy, off, w.n_theta, w.n_rho, np.float32(2) * np.float32(w.rho_max), w.threshold, w.window, t[0], t[1],
                           conformal_scale=2, want_circles=True)
    assert np.array_equal(ra.peaks, rb.peaks) and ca.tobytes() == cb.tobytes()
    # and with scale 2 the printed form holds literally: x_c = cos/rho_c, r_c = 1/|rho_c|
    q = int(ra.counts[0, 0]) - 1
    j, k = int(rb.peaks[0, q, 0]), int(rb.peaks[0, q, 1])
    rho_c = (k + 0.5) / float(np.float32(w.n_rho / (2.0 * float(np.float32(2) * np.float32(w.rho_max))))) - float(np.float32(2) * np.float32(w.rho_max))
    assert cb[0, q]["r_c"] == pytest.approx(1.0 / abs(rho_c), rel=1e-12) and cb[0, q]["x_c"] == pytest.approx(float(t[0][j]) / rho_c, rel=1e-12)


def test_n1_association_counts_against_the_numpy_bin_model():
    w = si.config(0)
    xy, off, _ = si.generate(w, 3)
    t = si.trig_table(w.n_theta)
    r, c = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], want_circles=True)
    for e in range(3):
        h = xy[off[e]:off[e + 1]]
        bins = npm.bins_f32(h, t[0], t[1], w.rho_max, w.n_rho)
        for q in range(min(int(r.counts[e, 0]), 64)):
            j, k = int(r.peaks[e, q, 0]), int(r.peaks[e, q, 1])
            assoc = (bins[:, j] >= 0) & (np.abs(bins[:, j] - k) <= w.window)
            assert c[e, q]["n_hits"] == int(assoc.sum()) and c[e, q]["n_hits"] >= 1
            z = (t[0][j] * h[assoc, 1] - t[1][j] * h[assoc, 0]).astype(np.float32)
            rho_c = (k + 0.5) / 21376.0 - float(si.RHO_MAX)
            z = z if rho_c >= 0 else -z
            assert c[e, q]["charge"] == int(np.sign(int((z < 0).sum()) - int((z > 0).sum())))


# ---------------------------------------------------------------- N2: numpy restatement and invariants
def nms_numpy(A, thr, permille, radius, wrap=False):
    W = A.astype(np.int64).copy()
    nt, nr = W.shape
    thr_eff = max(thr, -(-permille * int(W.max()) // 1000))
    out = []
    while True:
        c = int(np.argmax(W))                       # first occurrence of the maximum in raster order
        j, k = divmod(c, nr)
        v = int(W[j, k])
        if v == 0 or v < thr_eff:
            return out
        out.append([j, k, v])
        for dj in range(-radius, radius + 1):
            for dk in range(-radius, radius + 1):
                jj, kk = j + dj, k + dk
                if not 0 <= kk < nr:
                    continue
                if not 0 <= jj < nt:
                    if not wrap:
                        continue
                    while jj < 0:
                        jj, kk = jj + nt, nr - 1 - kk
                    while jj >= nt:
                        jj, kk = jj - nt, nr - 1 - kk
                W[jj, kk] = 0


@pytest.mark.parametrize("wrap", [False, True])
def test_n2_against_numpy_restatement_and_invariants(wrap):
    rng = np.random.default_rng(4)
    cases = [rng.poisson(2.0, size=(rng.integers(2, 24), rng.integers(2, 24))).astype(np.uint32) for _ in range(25)]
    w = si.config(0)
    xy, off, _ = si.generate(w, 2)
    t = si.trig_table(w.n_theta)
    cases += list(oracle.run(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], want_accum=True).accum)
    for A in cases:
        for pm, rad in ((300, 1), (600, 2), (0, 0)):
            n, p = oracle.find_peaks_ex(A, 3, max_peaks=100000, peak_mode=1, rel_permille=pm, nms_radius=rad, theta_wrap=wrap)
            assert p.tolist() == nms_numpy(A, 3, pm, rad, wrap) and n == len(p)
            if n:
                v = p[:, 2].astype(int)
                assert np.all(np.diff(v) <= 0) and v.min() >= max(3, -(-pm * int(A.max()) // 1000))       # descending, above the threshold
                assert np.array_equal(A[p[:, 0], p[:, 1]], p[:, 2])                                       # votes are the cells' own
                dj = np.abs(p[:, None, 0].astype(int) - p[None, :, 0].astype(int))
                dk = np.abs(p[:, None, 1].astype(int) - p[None, :, 1].astype(int))
                near = (dj <= rad) & (dk <= rad)
                np.fill_diagonal(near, False)
                assert not near.any()                                                                  # suppressed neighbourhoods hold no later peak
            n1, p1 = oracle.find_peaks_ex(A, 3, max_peaks=2, peak_mode=1, rel_permille=pm, nms_radius=rad, theta_wrap=wrap)
            assert n1 == n and np.array_equal(p1, p[:2])                                               # truncation stores the first, counts all


# ---------------------------------------------------------------- N4a: wrapped 3x3 and windows against numpy
def test_n4a_wrapped_3x3_against_a_padded_array_restatement():
    rng = np.random.default_rng(6)
    for _ in range(30):
        A = rng.poisson(1.5, size=(rng.integers(1, 20), rng.integers(1, 20))).astype(np.int64)
        nt, nr = A.shape
        P = np.zeros((nt + 2, nr + 2), dtype=np.int64)
        P[1:-1, 1:-1] = A
        P[0, 1:-1] = A[-1, ::-1]                    # column -1 = last column upside down
        P[-1, 1:-1] = A[0, ::-1]
        exp = []
        for j in range(nt):
            for k in range(nr):
                a = A[j, k]
                if a < 2:
                    continue
                nb = P[j:j + 3, k:k + 3]
                before = [nb[0, 0], nb[0, 1], nb[0, 2], nb[1, 0]]
                after = [nb[1, 2], nb[2, 0], nb[2, 1], nb[2, 2]]
                if all(a > b for b in before) and all(a >= b for b in after):
                    exp.append([j, k, int(a)])
        assert oracle.find_peaks_ex(A.astype(np.uint32), 2, theta_wrap=True)[1].tolist() == exp


def test_n4a_window_wrap_against_a_dilation_restatement():
    w = si.config(0)
    xy, off, _ = si.generate(w, 6)
    t = si.trig_table(w.n_theta)
    for win in (1, 3):
        r, _ = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, 12, win, t[0], t[1], max_peaks=4096, theta_wrap=True)
        r0, _ = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, 12, win, t[0], t[1], max_peaks=4096, theta_wrap=False)
        more = 0
        for e in range(6):
            h = xy[off[e]:off[e + 1]]
            bins = npm.bins_f32(h, t[0], t[1], w.rho_max, w.n_rho)
            D = np.zeros((w.n_theta, w.n_rho), dtype=bool)
            for j, k, _v in r.peaks[e, :r.counts[e, 0]]:
                for dj in range(-win, win + 1):
                    jj, kk = int(j) + dj, int(k)
                    if jj < 0:
                        jj, kk = jj + w.n_theta, w.n_rho - 1 - kk
                    elif jj >= w.n_theta:
                        jj, kk = jj - w.n_theta, w.n_rho - 1 - kk
                    D[jj, max(0, kk - win):min(w.n_rho - 1, kk + win) + 1] = True
            assert np.array_equal(r.keep[off[e]:off[e + 1]], npm.keep_from_dilation(bins, D))
            more += int(r.keep[off[e]:off[e + 1]].sum()) - int(r0.keep[off[e]:off[e + 1]].sum())
        assert more >= 0


# ---------------------------------------------------------------- N4b: distance filter against numpy fp64
def test_n4b_against_numpy_and_limits():
    w = si.config(0)
    xy, off, truth = si.generate(w, 5)
    t = si.trig_table(w.n_theta)
    for tol in (0.5, 2.0, 10.0):
        r, c = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], keep_mode=1, keep_tol=tol, want_circles=True)
        for e in range(5):
            h = xy[off[e]:off[e + 1]].astype(np.float64)
            ns = min(int(r.counts[e, 0]), 64)
            keep = np.zeros(len(h), dtype=bool)
            for q in range(ns):
                d = np.sqrt((h[:, 0] - c[e, q]["x_c"]) ** 2 + (h[:, 1] - c[e, q]["y_c"]) ** 2)
                keep |= np.abs(d - c[e, q]["r_c"]) < tol
            assert np.array_equal(r.keep[off[e]:off[e + 1]], keep.astype(np.uint8))
    r_inf, _ = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], keep_mode=1, keep_tol=1e30)
    r_zero, _ = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], keep_mode=1, keep_tol=0.0)
    assert r_inf.keep.all() and not r_zero.keep.any() and np.all(r_inf.counts[:, 0] > 0)
    # a 10 mm road around the candidate circles (the bin-centre radius is only good to 2 R^2 drho/2, tens of mm) keeps
    # nearly all signal hits and removes most of the background
    r2, _ = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, t[0], t[1], keep_mode=1, keep_tol=10.0)
    assert r2.keep[truth == 1].mean() > 0.9 and r2.keep[truth == 0].mean() < 0.2
