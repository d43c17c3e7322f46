"""-m gpu: the rows SURVEY.md 8(f) marks NEXT, through the C ABI, against oracle.run_ex, element by element and bit for
bit (fp64 circle records included): N1 candidate circles, N2 relative threshold + iterative NMS, N3 the paper's
1000 x 1000 grid on a 16-CTA cluster, N4a theta wrap, N4b original-space distance filter, N4c per-stream host staging."""
import numpy as np
import pytest

import oracle
import stcf_inputs as si
from tests.test_parity_gpu import compare

pytestmark = pytest.mark.gpu

OPTS = ("peak_mode", "rel_permille", "nms_radius", "theta_wrap", "keep_mode", "keep_tol", "b_field")
GPU_ONLY = ("staging", "scheduler", "select_mode")          # same results by definition: the oracle has no such options


@pytest.fixture(scope="module")
def hb():
    import torch
    assert torch.cuda.is_available()
    import paper_2607_04067_b200 as m
    m.load_library()
    return m


def gpu_ex(hb, w, xy, off, accum=True, circles=False, cluster_size=0, rho_max=None, **kw):
    import torch
    table = si.trig_table(w.n_theta)
    base = dict(max_peaks=w.max_peaks, acc_dtype=w.acc_dtype, threshold=w.threshold, window=w.window, conformal_scale=1)
    base.update({k: kw.pop(k) for k in list(kw) if k in base})
    opts = {k: kw.pop(k) for k in list(kw) if k in OPTS}
    gpu_only = {k: kw.pop(k) for k in list(kw) if k in GPU_ONLY}
    assert not kw, kw
    rho_max = w.rho_max if rho_max is None else rho_max
    h = hb.Hough(w.n_theta, w.n_rho, rho_max, base["threshold"], base["window"], max_peaks=base["max_peaks"], acc_dtype=base["acc_dtype"],
                 conformal_scale=base["conformal_scale"], cluster_size=cluster_size, trig_table=table, **opts, **gpu_only)
    try:
        d_xy = torch.from_numpy(np.ascontiguousarray(xy, dtype=np.float32).reshape(-1, 2)).cuda()
        d_off = torch.from_numpy(np.ascontiguousarray(off, dtype=np.int32)).cuda()
        out = h.alloc_outputs(d_xy.shape[0], d_off.numel() - 1, accum=accum)
        out["keep"].fill_(7); out["counts"].fill_(-99); out["kept_idx"].fill_(-5); out["peaks"].fill_(-1)
        h.run(d_xy, d_off, out=out)
        circ = h.circles(d_xy, d_off, out) if circles else None
        torch.cuda.synchronize()
        g = {k: v.cpu().numpy() for k, v in out.items()}
        g["peaks3"] = hb.unpack_peaks(g["peaks"])
        g["info"] = {"CLUSTER_SIZE": h.info(hb.HOUGH_INFO_CLUSTER_SIZE), "THREADS": h.info(hb.HOUGH_INFO_THREADS)}
        if circ is not None:
            g["circles"] = np.ascontiguousarray(circ.cpu().numpy()).view(hb.circle_dtype()).reshape(len(off) - 1, base["max_peaks"])
    finally:
        h.close()
    o, oc = oracle.run_ex(xy, off, w.n_theta, w.n_rho, rho_max, base["threshold"], base["window"], table[0], table[1],
                          max_peaks=base["max_peaks"], conformal_scale=base["conformal_scale"], acc_u16=(base["acc_dtype"] != "u32"),
                          want_accum=accum, n_threads=8, want_circles=circles, **opts)
    compare(g, o, off, base["max_peaks"], accum=accum, tag=w.name)
    if circles:
        for e in range(len(off) - 1):
            ns = min(int(o.counts[e, 0]), base["max_peaks"])
            assert g["circles"][e, :ns].tobytes() == oc[e, :ns].tobytes(), "circles of event %d" % e
            assert not np.frombuffer(g["circles"][e, ns:].tobytes(), dtype=np.uint8).any()      # entries past the stored ones are untouched
    return g, o, oc


def seam_events(w, n_ev):
    """Config-0 events with a noiseless track on the theta seam (centre direction 179.8 deg) added to the first one."""
    xy, off, _ = si.generate(w, n_ev)
    r = 200.0 + np.arange(48) * 600.0 / 47.0
    phi = np.deg2rad(179.8) - np.arccos(r / 1200.0)
    xy = np.concatenate([np.stack([r * np.cos(phi), r * np.sin(phi)], axis=1).astype(np.float32), xy])
    off = off.copy()
    off[1:] += 48
    return xy, off


# ---------------------------------------------------------------- N1
@pytest.mark.parametrize("cfg,n_ev", [(0, 16), (1, 60), (2, 8), (3, 4)])
def test_n1_circles_match_the_oracle_bit_for_bit(hb, cfg, n_ev):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    g, o, oc = gpu_ex(hb, w, xy, off, circles=True, accum=False)
    assert o.counts[:, 0].max() >= 1


def test_n1_closed_form_worked_example_scale_2_and_b_field(hb):
    # P1 on the GPU: r_c = 1644.31 mm, pT = 0.4933 GeV, charge and phi0 of either turning sense (tests/test_oracle_next_pins.py)
    from tests.test_oracle_next_pins import p1_hits
    w = si.config(0)
    for q in (1, -1):
        xy, R, phi_c = p1_hits(q)
        g, o, oc = gpu_ex(hb, w, xy, np.array([0, 48], dtype=np.int32), circles=True)
        i = g["peaks3"][0, :g["counts"][0, 0]].tolist().index([40, 70, 48])
        c = g["circles"][0, i]
        assert c["r_c"] == pytest.approx(1644.31, abs=0.01) and c["pt"] == pytest.approx(0.4933, abs=1e-4) and c["charge"] == q
        assert c["phi0"] == pytest.approx((phi_c - q * np.pi / 2) % (2 * np.pi), abs=1e-9)
    xy, off, _ = si.generate(w, 6)
    a, _, _ = gpu_ex(hb, w, xy, off, circles=True, b_field=0.5)
    b, _, _ = gpu_ex(hb, w, xy, off, circles=True, b_field=0.5, conformal_scale=2, rho_max=float(np.float32(2) * np.float32(w.rho_max)))
    assert a["circles"].tobytes() == b["circles"].tobytes()
    # W1 (tests/golden/w1_next.txt)
    w1 = type(w)(**{**w.__dict__, "n_theta": 4, "n_rho": 8, "rho_max": 2.0, "threshold": 2, "window": 0, "max_peaks": 8})
    xy1 = np.array([[1, 0], [0, 1], [.5, .5], [-1, 0], [0, 0], [4, 0]], dtype=np.float32)
    g, _, _ = gpu_ex(hb, w1, xy1, np.array([0, 6], dtype=np.int32), circles=True)
    assert [int(c) for c in g["circles"][0, :3]["charge"]] == [-1, -1, 1] and [int(c) for c in g["circles"][0, :3]["n_hits"]] == [2, 2, 3]
    assert g["circles"][0, 2]["r_c"] == 2.0 and g["circles"][0, 2]["phi0"] == 0.0


def test_n1_on_a_cluster_grid_and_with_empty_and_refused_events(hb):
    w = si.config(5)
    xy, off, _ = si.generate(w, 8)
    off2 = np.concatenate([[0, 0], off[1:]]).astype(np.int32)         # an empty event in front
    gpu_ex(hb, w, xy, off2, circles=True, accum=False)


# ---------------------------------------------------------------- N2
@pytest.mark.parametrize("cfg,n_ev,permille,radius", [(0, 16, 500, 1), (1, 64, 300, 2), (2, 6, 400, 1), (3, 4, 700, 3), (1, 20, 0, 0), (1, 20, 1000, 5)])
def test_n2_relative_threshold_and_iterative_nms(hb, cfg, n_ev, permille, radius):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    g, o, _ = gpu_ex(hb, w, xy, off, peak_mode=1, rel_permille=permille, nms_radius=radius)
    assert o.counts[:, 0].max() >= 1
    gpu_ex(hb, w, xy, off, peak_mode=1, rel_permille=permille, nms_radius=radius, max_peaks=3, accum=False)     # truncation


def test_n2_full_batch_of_1000_events(hb):
    w = si.config(1)
    xy, off, _ = si.generate(w)
    gpu_ex(hb, w, xy, off, peak_mode=1, rel_permille=500, nms_radius=2, accum=False)


def test_n2_with_theta_wrap_and_on_cluster_grids(hb):
    w0 = si.config(0)
    xy, off = seam_events(w0, 4)
    gpu_ex(hb, w0, xy, off, peak_mode=1, rel_permille=300, nms_radius=2, theta_wrap=True, threshold=12)
    # theta columns split over a cluster: one cluster barrier per extracted peak, the same decision in every CTA
    w5 = si.config(5)
    xy, off, _ = si.generate(w5, 2)
    gpu_ex(hb, w5, xy, off, peak_mode=1, rel_permille=400, nms_radius=2)
    xy, off = seam_events(w0, 4)
    xy, off = seam_events(w0, 2)
    for cluster in (2, 8):
        gpu_ex(hb, w0, xy, off, peak_mode=1, rel_permille=300, nms_radius=3, theta_wrap=True, threshold=12, cluster_size=cluster, circles=True)


# ---------------------------------------------------------------- N3
def test_n3_the_papers_1000x1000_grid_on_a_16_cta_cluster(hb):
    # rho in [-0.01, 0.01] (1/mm: 2/r at r = 200 mm, the scale of Eq. (2)), theta in [0, pi), 1000 bins each
    w = si.config(1)
    w = type(w)(**{**w.__dict__, "n_theta": 1000, "n_rho": 1000, "rho_max": 0.01, "threshold": 12, "window": 2, "max_peaks": 64})
    xy, off, _ = si.generate(w, 12)
    try:
        g, o, _ = gpu_ex(hb, w, xy, off, conformal_scale=2, circles=True)
    except hb.HoughError as e:
        if "16-CTA cluster" in str(e):      # cudaOccupancyMaxActiveClusters: this device cannot host a non-portable cluster
            pytest.skip(str(e))
        raise
    assert g["info"]["CLUSTER_SIZE"] == 16 and o.counts[:, 0].min() >= 1
    gpu_ex(hb, w, xy, off, conformal_scale=2, theta_wrap=True, keep_mode=1, keep_tol=3.0, accum=False)
    # the paper's own peak finder on the paper's own grid
    gpu_ex(hb, w, xy[:off[3]], off[:4], conformal_scale=2, peak_mode=1, rel_permille=500, nms_radius=3, theta_wrap=True, circles=True)


# ---------------------------------------------------------------- N4a / N4b
@pytest.mark.parametrize("cluster,window", [(0, 1), (0, 3), (2, 2), (8, 1)])
def test_n4a_theta_wrap(hb, cluster, window):
    w = si.config(0)
    xy, off = seam_events(w, 8)
    g, o, _ = gpu_ex(hb, w, xy, off, theta_wrap=True, window=window, threshold=12, max_peaks=512, cluster_size=cluster)
    o0, _ = oracle.run_ex(xy, off, w.n_theta, w.n_rho, w.rho_max, 12, window, *si.trig_table(w.n_theta), max_peaks=512)
    assert not np.array_equal(o.counts, o0.counts)                    # the seam track's mirrored duplicate peak is gone


@pytest.mark.parametrize("cfg,n_ev,cluster,tol", [(0, 16, 0, 5.0), (1, 40, 0, 2.0), (1, 12, 4, 20.0), (2, 4, 0, 1.0), (3, 3, 0, 0.5), (0, 4, 0, 0.0)])
def test_n4b_distance_filter(hb, cfg, n_ev, cluster, tol):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    gpu_ex(hb, w, xy, off, keep_mode=1, keep_tol=tol, cluster_size=cluster, accum=False)


def test_n4b_more_stored_peaks_than_staged_circles(hb):
    # a cluster stages only ~350 circles beside its compaction scratch: peaks beyond that come straight from the peak list
    w = si.config(3)
    xy, off, _ = si.generate(w, 2)
    g, o, _ = gpu_ex(hb, w, xy, off, keep_mode=1, keep_tol=0.2, cluster_size=2, accum=False)
    assert o.counts[:, 0].min() > 400


def test_option_validation(hb):
    h = hb.Hough(180, 128, 0.003, 10, 1)
    for key, bad in ((hb.HOUGH_OPT_PEAK_MODE, 2), (hb.HOUGH_OPT_REL_THRESHOLD_PERMILLE, 1001), (hb.HOUGH_OPT_NMS_RADIUS, 65),
                     (hb.HOUGH_OPT_THETA_WRAP, 2), (hb.HOUGH_OPT_KEEP_MODE, -1), (hb.HOUGH_OPT_CLUSTER_SIZE, 3)):
        with pytest.raises(hb.HoughError):
            hb.hough_set_option(h.ctx, key, bad)
    with pytest.raises(hb.HoughError):
        hb.hough_set_option_f64(h.ctx, hb.HOUGH_OPTF_KEEP_TOL, -1.0)
    with pytest.raises(hb.HoughError):
        hb.hough_set_option_f64(h.ctx, 99, 1.0)
    h.close()


# ---------------------------------------------------------------- N4c: sub-batches on several streams, one staging area each
def test_n4c_host_sub_batches_on_several_streams_overlap_safely(hb):
    import torch
    w = si.config(1)
    xy, off, _ = si.generate(w, 200)
    table = si.trig_table(w.n_theta)
    o = oracle.run(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table[0], table[1], max_peaks=w.max_peaks, n_threads=8)
    h = hb.Hough(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, trig_table=table)
    h_xy, h_off = torch.from_numpy(xy).pin_memory(), torch.from_numpy(off).pin_memory()
    keep = torch.full((len(xy),), 9, dtype=torch.uint8).pin_memory()
    peaks = torch.zeros((200, 64, 2), dtype=torch.int32).pin_memory()
    counts = torch.full((200, 2), -7, dtype=torch.int32).pin_memory()
    kxy = torch.zeros((len(xy), 2), dtype=torch.float32).pin_memory()
    kidx = torch.full((len(xy),), -3, dtype=torch.int32).pin_memory()
    streams = [torch.cuda.Stream() for _ in range(4)]
    for rep in range(2):                                   # the second pass reuses every stream's staging area
        for b, e0 in enumerate(range(0, 200, 25)):         # 8 sub-batches of 25 events, round-robin on 4 streams
            hb.hough_run_host(h.ctx, h_xy, h_off[e0:], 25, keep, peaks[e0:], counts[e0:], kxy, kidx, stream=streams[b % 4])
        torch.cuda.synchronize()
        assert np.array_equal(counts.numpy(), o.counts) and np.array_equal(keep.numpy(), o.keep)
        p3 = hb.unpack_peaks(peaks.numpy())
        for e in range(200):
            ns = min(int(o.counts[e, 0]), 64)
            assert np.array_equal(p3[e, :ns], o.peaks[e, :ns]) and not p3[e, ns:].any()
            nk, a = int(o.counts[e, 1]), int(off[e])
            assert np.array_equal(kidx.numpy()[a:a + nk], o.kept_idx[a:a + nk])
            assert np.array_equal(kxy.numpy()[a:a + nk].view(np.uint32), o.kept_xy[a:a + nk].view(np.uint32))
            assert not kidx.numpy()[a + nk:int(off[e + 1])].any()          # the tail comes back zeroed
    # more streams than staging slots: the least recently used slot is recycled
    many = [torch.cuda.Stream() for _ in range(10)]
    for b, e0 in enumerate(range(0, 200, 20)):
        hb.hough_run_host(h.ctx, h_xy, h_off[e0:], 20, keep, peaks[e0:], counts[e0:], None, None, stream=many[b])
    torch.cuda.synchronize()
    assert np.array_equal(counts.numpy(), o.counts) and np.array_equal(keep.numpy(), o.keep)
    h.close()


# ---------------------------------------------------------------- H0 variant: bulk-copy (TMA engine) staging.  Kept last in the
# file: it is the one path whose PTX (cp.async.bulk + mbarrier) has no CPU restatement beyond a memcpy.  The wait on the
# mbarrier is bounded in the kernel, so a mistake shows up as a mismatch, never as a hang.
@pytest.mark.parametrize("cfg,n_ev,cluster", [(0, 16, 0), (1, 100, 0), (3, 6, 0), (5, 12, 0), (1, 30, 4)])
def test_h0_bulk_copy_staging(hb, cfg, n_ev, cluster):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    gpu_ex(hb, w, xy, off, staging=1, cluster_size=cluster)
    # without the batch's first hit every event starts at the other parity and the batch ends on the other parity
    gpu_ex(hb, w, np.ascontiguousarray(xy[1:]), np.concatenate([[0], off[1:] - 1]).astype(np.int32), staging=1, cluster_size=cluster, accum=False)


def test_h0_bulk_copy_staging_chunked_events_and_alignment_check(hb):
    import torch
    w3 = si.config(3)
    xy3, off3, _ = si.generate(w3, 6)
    big = np.ascontiguousarray(xy3[1:off3[6]])                       # ~17000 hits in one event: several copies, each with its own shift
    gpu_ex(hb, w3, big, np.array([0, 5, len(big)], dtype=np.int32), staging=1, threshold=60)
    w = si.config(0)
    xy, off, _ = si.generate(w, 4)
    h = hb.Hough(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, staging=1)
    d = torch.from_numpy(np.concatenate([xy[:1], xy])).cuda()      # a view that starts 8 bytes into the allocation
    out = h.alloc_outputs(len(xy), 4)
    with pytest.raises(hb.HoughError, match="16-byte"):
        hb.hough_run(h.ctx, d[1:], torch.from_numpy(off).cuda(), 4, out["keep"], out["peaks"], out["counts"])
    h.close()


# ---------------------------------------------------------------- scheduler variant: persistent CTAs that steal not-yet-launched
# CTAs' events (cluster launch control) and prefetch the next event's hits into L2.  Bounded waits: a mistake is a mismatch.
@pytest.mark.parametrize("cfg,n_ev,staging", [(0, 16, 0), (1, 1000, 0), (1, 400, 1), (2, 300, 0), (3, 200, 1)])
def test_work_stealing_scheduler(hb, cfg, n_ev, staging):
    # more events than resident CTA slots (296 for the 180 x 256 u16 grid), so that requests succeed AND fail
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    gpu_ex(hb, w, xy, off, scheduler=1, staging=staging, accum=False)


def test_work_stealing_scheduler_with_empty_refused_and_chunked_events_and_on_streams(hb):
    import torch
    w = si.config(1)
    xy, off, _ = si.generate(w, 600)
    off2 = np.concatenate([[0, 0], off[1:300], [off[299]], off[300:]]).astype(np.int32)        # empty events in between
    gpu_ex(hb, w, xy, off2, scheduler=1, accum=False)
    w3 = si.config(3)
    xy3, off3, _ = si.generate(w3, 400)
    cut = int(off3[6])
    off_big = np.concatenate([[0, cut], off3[7:]]).astype(np.int32)                            # the first event has ~17000 hits
    gpu_ex(hb, w3, xy3, off_big, scheduler=1, threshold=60, accum=False)
    # the same handle on three streams at once (no scratch, no counter: the requests of different launches never mix)
    table = si.trig_table(w.n_theta)
    o = oracle.run(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table[0], table[1], max_peaks=w.max_peaks, n_threads=8)
    h = hb.Hough(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, trig_table=table, scheduler=1)
    d_xy, d_off = torch.from_numpy(xy).cuda(), torch.from_numpy(off).cuda()
    outs, streams = [], [torch.cuda.Stream() for _ in range(3)]
    torch.cuda.synchronize()
    for s in streams:
        outs.append(h.run(d_xy, d_off, stream=s, kept=False))
    torch.cuda.synchronize()
    for out in outs:
        assert np.array_equal(out["counts"].cpu().numpy(), o.counts) and np.array_equal(out["keep"].cpu().numpy(), o.keep)
    h.close()


# ---------------------------------------------------------------- H6 variant: dense selection (the accumulator rewritten as the
# window mask, every hit tested at all columns with the voting loop's mapping).  Same results by definition.
@pytest.mark.parametrize("cfg,n_ev,mode,extra", [(0, 16, 1, {}), (1, 40, 1, {}), (2, 24, 1, {}), (3, 12, 1, {}), (2, 12, 2, {}), (1, 30, 2, {}),
                                                 (5, 8, 1, {}), (0, 16, 1, dict(theta_wrap=True)), (3, 8, 1, dict(peak_mode=1, rel_permille=300, window=1)),
                                                 (1, 20, 1, dict(staging=1, scheduler=1))])
def test_h6_dense_selection(hb, cfg, n_ev, mode, extra):
    w = si.config(cfg)
    xy, off, _ = si.generate(w, n_ev)
    gpu_ex(hb, w, xy, off, select_mode=mode, accum=False, **extra)


def test_h6_dense_selection_with_degenerate_hits_chunked_events_and_more_hits_than_flag_bits(hb):
    w = si.config(0)
    xy, off, _ = si.generate(w, 3)
    bad = np.array([[0, 0], [np.inf, 1], [1e-3, 0], [1e-20, 1e-20], [np.nan, 5], [1e30, 1e30], [3e38, 0]], dtype=np.float32)
    xy2 = np.concatenate([xy[:off[1]], bad, xy[off[1]:]])
    off2 = np.concatenate([[0, 0], off[1:2] + len(bad), off[2:] + len(bad), [off[-1] + len(bad)]]).astype(np.int32)
    gpu_ex(hb, w, xy2, off2, select_mode=1, threshold=5, accum=False)
    w3 = si.config(3)
    xy3, off3, _ = si.generate(w3, 12)
    cut = int(off3[6])                                                # ~17000 hits in one event: chunked, and more hits than the bitmap has bits
    gpu_ex(hb, w3, xy3[:off3[12]], np.concatenate([[0, cut], off3[7:13]]).astype(np.int32), select_mode=1, threshold=60, accum=False)
