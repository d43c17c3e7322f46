#!/usr/bin/env python
"""bench.py -- throughput of the conformal Hough hot path (H0-H7) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic events
(default: BASELINE.json configs[1], the 1000-event nominal-background batch,
regenerated from its seed): ONE hough_run() launch through the C ABI.  Rank 0
prints ONE JSON line (contract in DESIGN.md "Measurement").

  value / ms_per_step : events/s with inputs and outputs resident in HBM; every
                        step is timed by its own CUDA-event pair on the launching
                        stream and L2 is flushed (256 MiB write) before each step
  e2e                 : the same metric through hough_run_host() with pinned HOST
                        buffers: H2D of hits+offsets and D2H of the results inside
                        the timed region
                        (lean: mask + peaks + counts come back; e2e.full adds the
                        compacted hits)
  roofline            : achieved in-range votes/s of the one kernel against the
                        shared-atomic rate measured live on this GPU, plus the
                        HBM term (north_star: the slower of the two binds)
  all_configs         : events/s, Gvotes/s and roofline fraction of EVERY BASELINE.json
                        configuration (0-3, the 100k-event sweep at 180x256 and at the
                        360x512 cluster grid), >= 20 CUDA-event-timed steps each
  multi_stream        : the sweep in batches of 1k/10k/100k events on 1/2/4 streams
  cpu_baseline        : the oracle, as it stands, on the host cores (rank 0, N=1)

--impl reference times the oracle (the only reference this tier has) and is
the one other place that executes oracle/.  Under torchrun every rank works on
its own events (weak scaling, no data-path collective: events are independent,
PAPER.md:88-90); the time is the max over ranks.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/s (1000-event batch; Gvotes/s = hit x theta pairs, and % of roofline, in the same line)"
UNIT = "events/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=1, help="index into stcf_inputs.CONFIGS (1 = nominal 1000 events)")
    ap.add_argument("--events", type=int, default=0, help="override the number of events per rank")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-flush", action="store_true", help="do not flush L2 between steps (diagnostic only)")
    ap.add_argument("--ctas-per-sm", type=int, default=0)
    ap.add_argument("--cluster", type=int, default=0)
    ap.add_argument("--vote-path", type=int, default=0,
                    help="HOUGH_OPT_VOTE_PATH (0 packed fast, 1 exact slow; 2/3 = phase-skipping diagnostics of the bench-only diag build)")
    ap.add_argument("--staging", type=int, default=0, help="HOUGH_OPT_STAGING (0 coalesced loads, 1 cp.async.bulk per chunk)")
    ap.add_argument("--scheduler", type=int, default=0, help="HOUGH_OPT_SCHEDULER (0 one CTA per event, 1 work stealing by cluster launch control)")
    ap.add_argument("--select", type=int, default=0, help="HOUGH_OPT_SELECT_MODE (0 scan of the marked columns, 1 dense, 2 dense when many peaks)")
    ap.add_argument("--no-all-configs", action="store_true", help="skip the all_configs / multi_stream blocks (headline only)")
    ap.add_argument("--config-steps", type=int, default=20, help="timed steps per configuration in the all_configs block")
    ap.add_argument("--sweep-events", type=int, default=100000, help="events of the config-4 sweep (all_configs, multi_stream)")
    ap.add_argument("--segment", default="", choices=["", "probes"],
                    help="internal: run one side measurement in this (child) process and print its JSON")
    return ap.parse_args()


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


# ---------------------------------------------------------------- clocks during the timed region
class ClockSampler:
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, dev):
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop = threading.Event()
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:      # the torch device, whatever CUDA_VISIBLE_DEVICES says
                self.h = pynvml.nvmlDeviceGetHandleByUUID("GPU-" + str(torch.cuda.get_device_properties(dev).uuid))
            except Exception:  # noqa: BLE001
                self.h = pynvml.nvmlDeviceGetHandleByIndex(dev.index or 0)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # noqa: BLE001 -- NVML missing: report it in the line
            self.err = str(e)
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:  # noqa: BLE001
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:  # noqa: BLE001
                pass
            time.sleep(0.002)

    def start(self):
        if self.ok:
            self.t.start()

    def stop(self):
        self._stop.set()
        if self.ok:
            self.t.join()
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# ---------------------------------------------------------------- the reference arm = the oracle on the host cores
def oracle_rate(w, xy, off, n_sample, n_threads, reps):
    """events/s of oracle.run on the first n_sample events, `reps` passes, n_threads host threads."""
    import oracle
    import stcf_inputs as si
    table = si.trig_table(w.n_theta)
    o2 = off[:n_sample + 1]
    x2 = xy[:int(o2[-1])]
    t0 = time.perf_counter()
    for _ in range(reps):
        oracle.run(x2, o2, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, table[0], table[1],
                   max_peaks=w.max_peaks, acc_u16=(w.acc_dtype != "u32"), n_threads=n_threads)
    dt = time.perf_counter() - t0
    return n_sample * reps / dt, dt


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    import stcf_inputs as si
    w = si.config(args.config)
    n_events = args.events or min(w.n_events, 1000)
    xy, off, _ = si.generate(w, n_events)
    cores = len(os.sched_getaffinity(0))
    # size the per-step sample so that the whole run stays within about a minute
    probe_n = min(64, n_events)
    rate, _ = oracle_rate(w, xy, off, probe_n, cores, 1)
    budget_s = 60.0
    n_sample = int(max(8, min(n_events, rate * budget_s / max(1, args.steps + args.warmup))))
    for _ in range(args.warmup):
        oracle_rate(w, xy, off, n_sample, cores, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_rate(w, xy, off, n_sample, cores, 1)
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    n_hits = int(off[n_sample])
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(w, n_events, 1, extra={"sample_events_per_step": n_sample}),
        "gvotes_per_s": n_hits * w.n_theta * args.steps / dt / 1e9,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "first %d events of the batch per step, %d steps, %d threads (one event range per thread)"
                                   % (n_sample, args.steps, cores)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(w, n_events, world, extra=None):
    c = {
        "workload": "%s: %d events/GPU x %d GPU(s), seed %d, N_theta=%d, N_rho=%d, %s accumulator, threshold %d, window %d, max_peaks %d"
                    % (w.name, n_events, world, w.seed, w.n_theta, w.n_rho, w.acc_dtype, w.threshold, w.window, w.max_peaks),
        "events_per_gpu": n_events, "n_theta": w.n_theta, "n_rho": w.n_rho, "acc_dtype": w.acc_dtype,
        "threshold": w.threshold, "window": w.window, "max_peaks": w.max_peaks,
        "parallelism": "events sharded across ranks, no collective" if world > 1 else "single GPU",
    }
    if extra:
        c.update(extra)
    return c


# ---------------------------------------------------------------- our arm
def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:  # noqa: BLE001
        return 6650.0, "fallback (B200_PROFILING.md)"


def run_probe_segment():
    """Child process of device_probes(): the two measurement aids of include/hough_bench.h on this rank's GPU, each
    guarded, one JSON object on stdout."""
    import torch
    import paper_2607_04067_b200 as hb
    _, local_rank, _ = dist_env()
    torch.cuda.set_device(local_rank)
    torch.zeros(1, device=torch.device("cuda", local_rank))
    out = {}
    for key, call in (("atom_rate", lambda: hb.hough_bench_shared_atomics(5, 1, 1024, 20000)),      # conflict-free ATOMS/s, all SMs
                      ("vote_loop", lambda: hb.hough_bench_vote_loop(15, 6, 2, 512, 20))):          # the voting loop's instruction sequence alone
        try:
            out[key] = float(call())
        except Exception as ex:  # noqa: BLE001
            out[key + "_error"] = "%s: %s" % (type(ex).__name__, ex)
    print(json.dumps(out), flush=True)
    return 0


def device_probes(sm_count, sm_max_mhz, timeout_s=300):
    """The roofline's denominator (hough_bench_shared_atomics(5)) and the vote-loop probe, measured now, in a process
    of their own: the measurement aids are not product code, and a failure in them (even one that loses the CUDA
    context) must not cost the headline.  If the measurement fails the peak is the derived one -- 32 shared atomics
    per clock per SM (one per lane per issue) x SMs x the maximum SM clock -- and says so."""
    import subprocess
    res, err = {}, None
    try:
        r = subprocess.run([sys.executable, os.path.abspath(__file__), "--segment", "probes"], capture_output=True, text=True,
                           timeout=timeout_s, cwd=ROOT)
        lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
        if lines:
            res = json.loads(lines[-1])
        else:
            err = "probe process exited %s: %s" % (r.returncode, (r.stderr or "").strip().splitlines()[-1:] or "no output")
    except Exception as ex:  # noqa: BLE001
        err = "%s: %s" % (type(ex).__name__, ex)
    atom_rate, probe = res.get("atom_rate"), res.get("vote_loop")
    if atom_rate and atom_rate > 0:
        src = "hough_bench_shared_atomics(variant 5) measured in this run: conflict-free 32-bit shared atomics, all SMs"
    else:
        atom_rate = 32.0 * (sm_count or 148) * (sm_max_mhz or 1965) * 1e6
        src = ("DERIVED, not measured: 32 shared atomics per clock per SM x %d SMs x %d MHz (the live measurement failed: %s)"
               % (sm_count or 148, sm_max_mhz or 1965, err or res.get("atom_rate_error")))
    return atom_rate, src, (probe if probe and probe > 0 else None), (None if probe else err or res.get("vote_loop_error"))


class Workbench:
    """One workload resident on the device: inputs, outputs, handle.  Marshalling and timing only."""

    def __init__(self, hb, si, torch, dev, cfg, n_events, first_event=0, cluster=0, ctas_per_sm=0, vote_path=0, staging=0, scheduler=0, select=0):
        self.hb, self.torch, self.dev = hb, torch, dev
        self.w = w = si.config(cfg)
        self.n_events = n_events
        self.xy, self.off, self.truth = si.generate(w, n_events, first_event=first_event)
        self.n_total = len(self.xy)
        self.table = si.trig_table(w.n_theta)
        self.h = hb.Hough(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, max_peaks=w.max_peaks, acc_dtype=w.acc_dtype,
                          cluster_size=cluster, ctas_per_sm=ctas_per_sm, trig_table=self.table, staging=staging, scheduler=scheduler, select_mode=select)
        if vote_path:
            hb.hough_set_option(self.h.ctx, hb.HOUGH_OPT_VOTE_PATH, vote_path)
        self.info = {k: self.h.info(getattr(hb, "HOUGH_INFO_" + k)) for k in
                     ("CLUSTER_SIZE", "THREADS", "SMEM_BYTES", "CTAS_PER_SM", "GRID_MAX", "ACC_BITS", "CHUNK_HITS", "SM_COUNT")}
        self.d_xy = torch.from_numpy(self.xy).to(dev)
        self.d_off = torch.from_numpy(self.off).to(dev)
        self.out = self.h.alloc_outputs(self.n_total, n_events, dev, kept=True, accum=False)
        self.pairs = self.n_total * w.n_theta

    def step(self, stream):
        o = self.out
        self.hb.hough_run_ex(self.h.ctx, self.d_xy, self.d_off, self.n_events, o["keep"], o["peaks"], o["counts"],
                             o["kept_xy"], o["kept_idx"], None, stream)

    def timed(self, steps, warmup, flush, stream):
        """`steps` launches, each with its own CUDA-event pair on the launching stream (ms per step)."""
        torch = self.torch
        for _ in range(max(warmup, 3)):
            if flush is not None:
                flush.zero_()
            self.step(stream)
        torch.cuda.synchronize()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in evs:
            if flush is not None:
                flush.zero_()
            a.record(stream)
            self.step(stream)
            b.record(stream)
        torch.cuda.synchronize()
        import numpy as np
        return np.array([a.elapsed_time(b) for a, b in evs], dtype=np.float64)

    def in_range_votes(self, sample_events=None):
        """V_in = sum of all accumulator cells (one shared atomic per in-range vote: the roofline's unit), from the
        kernel's own dump, untimed.  With sample_events the fraction of a leading sample is scaled to the batch."""
        torch = self.torch
        n_ev = self.n_events if sample_events is None else min(sample_events, self.n_events)
        v_in, step_ev = 0, 125
        for e0 in range(0, n_ev, step_ev):
            e1 = min(n_ev, e0 + step_ev)
            sub_off = (self.d_off[e0:e1 + 1] - self.d_off[e0]).contiguous()
            sub_xy = self.d_xy[int(self.off[e0]):int(self.off[e1])]
            o = self.h.run(sub_xy, sub_off, kept=False, accum=True)
            v_in += int(o["accum"].sum(dtype=torch.int64).item())
            del o
        if n_ev == self.n_events:
            return v_in, "exact"
        frac = v_in / max(1, int(self.off[n_ev]) * self.w.n_theta)
        return int(round(frac * self.pairs)), "in-range fraction of the first %d events x all pairs" % n_ev

    def counts(self):
        c = self.out["counts"].cpu()
        return int(c[:, 1].sum().item()), int(c[:, 0].clamp(max=self.w.max_peaks).sum().item())

    def retention(self):
        """The paper's two quality figures on the synthetic events (context, not a parity claim): data compression ratio
        R_c = N_select / N_total (Eq. (8)) and signal retention ratio R_s = N_true,select / N_true
        (Eq. (9)), N_true = the generator's signal-track hits."""
        keep = self.out["keep"].cpu().numpy().astype(bool)
        sig = self.truth.astype(bool)
        return {"R_c": float(keep.mean()) if keep.size else None, "R_s": float(keep[sig].mean()) if sig.any() else None,
                "signal_hit_fraction": float(sig.mean()) if sig.size else None}

    def alg_bytes(self, counts=None):
        n_kept, n_peaks = counts if counts is not None else self.counts()
        return 8 * self.n_total + 4 * (self.n_events + 1) + self.n_total + 12 * n_kept + 8 * n_peaks + 8 * self.n_events

    def close(self):
        self.h.close()


def roofline_block(wb, t_kernel_s, v_in, v_in_how, atom_rate, hbm_gbs, hbm_src, counts=None, atom_src=None):
    alg_bytes = wb.alg_bytes(counts)
    t_vote, t_hbm = v_in / atom_rate, alg_bytes / (hbm_gbs * 1e9)
    return {
        "bound": "alu", "pipe": "shared-memory atomics (ATOMS), one per in-range vote; the slower of the vote and HBM terms binds (north_star)",
        "achieved": v_in / t_kernel_s / 1e9, "peak": atom_rate / 1e9, "unit": "Gvotes/s (in-range)",
        "frac": max(t_vote, t_hbm) / t_kernel_s,
        "traffic": None, "traffic_note": "no ncu capture of this commit in this run; see profiles/ for the last one and its commit",
        "peak_source": atom_src or "hough_bench_shared_atomics(variant 5) measured in this run: conflict-free 32-bit shared atomics, all SMs",
        "algorithmic_votes_per_launch": v_in, "votes_counted": v_in_how, "algorithmic_bytes_per_launch": alg_bytes,
        "t_vote_us": t_vote * 1e6, "t_hbm_us": t_hbm * 1e6, "t_kernel_us": t_kernel_s * 1e6,
        "hbm": {"achieved": alg_bytes / t_kernel_s / 1e9, "peak": hbm_gbs, "unit": "GB/s", "frac": t_hbm / t_kernel_s, "peak_source": hbm_src},
    }


def config_line(wb, times_ms, v_in, v_in_how, atom_rate, hbm_gbs, hbm_src):
    import numpy as np
    ms = float(times_ms.mean())
    t = ms * 1e-3
    r = roofline_block(wb, t, v_in, v_in_how, atom_rate, hbm_gbs, hbm_src)
    n_kept, _ = wb.counts()
    return {"workload": wb.w.name, "events": wb.n_events, "hits": wb.n_total, "grid": "%dx%d %s" % (wb.w.n_theta, wb.w.n_rho, wb.w.acc_dtype),
            "cluster_size": wb.info["CLUSTER_SIZE"], "threads": wb.info["THREADS"], "ctas_per_sm": wb.info["CTAS_PER_SM"],
            "steps": int(len(times_ms)), "ms_per_step": ms, "ms_per_step_min": float(times_ms.min()), "ms_per_step_median": float(np.median(times_ms)),
            "events_per_s": wb.n_events / t, "gvotes_per_s": wb.pairs / t / 1e9, "gvotes_in_range_per_s": v_in / t / 1e9,
            "frac": r["frac"], "hbm_frac": r["hbm"]["frac"], "kept_fraction": n_kept / max(1, wb.n_total), "quality": wb.retention()}


def multi_stream_sweep(wb, torch, batches=(1000, 10000, 100000), streams_list=(1, 2, 4), reps=3):
    """BASELINE.json config 4: the sweep's events in batches of 1k / 10k / 100k on 1, 2 and 4 CUDA streams through ONE
    handle (no per-run scratch; PAPER.md:90 batching, :204-210 batch scaling).  A sub-batch is a pointer offset into
    the same device arrays (offsets are absolute), so nothing is copied.  Device time from a start event that every
    stream waits on to the last stream's end event."""
    hb, o = wb.hb, wb.out
    res = []
    pools = {n: [torch.cuda.Stream() for _ in range(n)] for n in streams_list}
    main = torch.cuda.current_stream()
    for B in batches:
        if B > wb.n_events:
            continue
        for ns in streams_list:
            st = pools[ns]
            best = None
            for rep in range(reps + 1):            # the first repetition is the warm-up
                torch.cuda.synchronize()
                start = torch.cuda.Event(enable_timing=True)
                ends = [torch.cuda.Event(enable_timing=True) for _ in st]
                start.record(main)
                for s_ in st:
                    s_.wait_event(start)
                for bi, e0 in enumerate(range(0, wb.n_events, B)):
                    e1 = min(wb.n_events, e0 + B)
                    hb.hough_run_ex(wb.h.ctx, wb.d_xy, wb.d_off[e0:], e1 - e0, o["keep"], o["peaks"][e0:], o["counts"][e0:],
                                    o["kept_xy"], o["kept_idx"], None, st[bi % ns])
                for s_, ev in zip(st, ends):
                    ev.record(s_)
                torch.cuda.synchronize()
                ms = max(start.elapsed_time(ev) for ev in ends)
                if rep > 0:
                    best = ms if best is None else min(best, ms)
            res.append({"batch_events": B, "streams": ns, "launches": (wb.n_events + B - 1) // B, "ms_total": best,
                        "events_per_s": wb.n_events / (best * 1e-3)})
    return res


def run_ours(args):
    import numpy as np
    import torch
    if args.vote_path >= 2:
        os.environ["HOUGH_B200_FLAVOR"] = "diag"     # the phase-skipping diagnostics live in a bench-only build
    import paper_2607_04067_b200 as hb
    import stcf_inputs as si
    from paper_2607_04067_b200 import shard

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    hb.load_library()   # raises if the CUDA library cannot be built / loaded
    w = si.config(args.config)
    n_events = args.events or min(w.n_events, 1000)
    first_event, _ = shard.event_range(rank, world, n_events)             # every rank its own events
    wb = Workbench(hb, si, torch, dev, args.config, n_events, first_event, args.cluster, args.ctas_per_sm, args.vote_path,
                   args.staging, args.scheduler, args.select)
    xy, off, n_total, info, h = wb.xy, wb.off, wb.n_total, dict(wb.info), wb.h
    info["VOTE_PATH"] = args.vote_path
    info["STAGING"], info["SCHEDULER"], info["SELECT_MODE"] = args.staging, args.scheduler, args.select      # 0 / 0 / 0 = the defaults
    info["LIBRARY"] = os.path.basename(hb.lib_path())
    stream = torch.cuda.current_stream()
    flush = None if args.no_flush else torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    # ---- the headline: `steps` timed launches, cold L2, clocks sampled during the timed region
    for _ in range(max(args.warmup, 3)):
        if flush is not None:
            flush.zero_()
        wb.step(stream)
    torch.cuda.synchronize()
    launches0 = h.info(hb.HOUGH_INFO_LAUNCHES)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(dev)
    barrier()
    torch.cuda.synchronize()
    sampler.start()
    t_wall0 = time.perf_counter()
    for a, b in evs:
        if flush is not None:
            flush.zero_()
        a.record(stream)
        wb.step(stream)
        b.record(stream)
    torch.cuda.synchronize()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    launches = h.info(hb.HOUGH_INFO_LAUNCHES) - launches0
    times = np.array([a.elapsed_time(b) for a, b in evs], dtype=np.float64)   # ms
    total_ms = float(times.sum())

    # back to back, warm L2 (diagnostic)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(args.steps):
        wb.step(stream)
    b.record(stream)
    torch.cuda.synchronize()
    warm_ms = a.elapsed_time(b) / args.steps

    # ---- what the roofline needs from the device, gathered before anything else runs (untimed)
    v_in, v_in_how = wb.in_range_votes(None if n_events <= 5000 else 2000)
    alg_counts = wb.counts()
    quality = wb.retention()
    # the measurement aids run in a process of their own (this one is idle meanwhile): see device_probes()
    atom_rate, atom_src, probe, probe_err = device_probes(info["SM_COUNT"], clocks.get("sm_max_mhz"))

    # ---- end to end through hough_run_host: pinned host buffers, copies inside the timed region.
    # "lean" (headline e2e): H2D hits + offsets, D2H mask + peaks + counts -- what a host consumer that still holds its
    # hits needs; "full" adds the compacted hits and their indices (full-length arrays, reading Q11).
    h_xy, h_off = torch.from_numpy(xy).pin_memory(), torch.from_numpy(off).pin_memory()
    h_keep = torch.empty(n_total, dtype=torch.uint8).pin_memory()
    h_peaks = torch.zeros((n_events, w.max_peaks, 2), dtype=torch.int32).pin_memory()
    h_counts = torch.empty((n_events, 2), dtype=torch.int32).pin_memory()
    h_kxy = torch.empty((n_total, 2), dtype=torch.float32).pin_memory()
    h_kidx = torch.empty(n_total, dtype=torch.int32).pin_memory()
    e2e_steps = min(args.steps, 50)
    e2e = {}
    e2e_err = {}
    for mode, kx, ki in (("lean", None, None), ("full", h_kxy, h_kidx)):
        ms_sum = 0.0
        try:      # an error here is reported in the line's e2e block; it must not cost the device-resident headline
            for _ in range(3):
                hb.hough_run_host(h.ctx, h_xy, h_off, n_events, h_keep, h_peaks, h_counts, kx, ki, stream)
            torch.cuda.synchronize()
            barrier()
            for _ in range(e2e_steps):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                hb.hough_run_host(h.ctx, h_xy, h_off, n_events, h_keep, h_peaks, h_counts, kx, ki, stream)
                b.record(stream)
                b.synchronize()               # the caller reads the results on the host here
                ms_sum += a.elapsed_time(b)
            barrier()
            # the host results must be the device-resident run's (same inputs): a cheap end-to-end sanity check, untimed
            if int(h_counts[:, 1].sum().item()) != alg_counts[0] or int(h_keep.sum().item()) != alg_counts[0]:
                raise RuntimeError("hough_run_host returned %d kept hits (mask %d), the device-resident run %d"
                                   % (int(h_counts[:, 1].sum().item()), int(h_keep.sum().item()), alg_counts[0]))
        except Exception as ex:  # noqa: BLE001
            if world > 1:
                raise                          # ranks must stay in step: no partial line under torchrun
            ms_sum, e2e_err[mode] = float("nan"), "%s: %s" % (type(ex).__name__, ex)
        d2h = h_keep.numel() + h_peaks.numel() * 4 + h_counts.numel() * 4 + (0 if kx is None else h_kxy.numel() * 4 + h_kidx.numel() * 4)
        e2e[mode] = (ms_sum, d2h)
    h2d = h_xy.numel() * 4 + h_off.numel() * 4
    # the same lean transfer as 4 sub-batches on 4 streams (one staging area per stream): copies overlap kernels
    ov_streams = [torch.cuda.Stream() for _ in range(4)]
    sub = (n_events + 3) // 4

    def overlapped():
        start = torch.cuda.Event(enable_timing=True)
        start.record(stream)
        ends = []
        for b_, s_ in enumerate(ov_streams):
            e0 = b_ * sub
            ne = min(sub, n_events - e0)
            if ne <= 0:
                continue
            s_.wait_event(start)
            hb.hough_run_host(h.ctx, h_xy, h_off[e0:], ne, h_keep, h_peaks[e0:], h_counts[e0:], None, None, s_)
            ev = torch.cuda.Event(enable_timing=True)
            ev.record(s_)
            ends.append(ev)
        torch.cuda.synchronize()
        return max(start.elapsed_time(ev) for ev in ends)

    e2e_ov_err = None
    try:
        for _ in range(3):
            overlapped()
        e2e_ov_ms = sum(overlapped() for _ in range(e2e_steps))
    except Exception as ex:  # noqa: BLE001 -- a side figure must not cost the line
        e2e_ov_ms, e2e_ov_err = float("nan"), "%s: %s" % (type(ex).__name__, ex)
    barrier()

    # ---- max over ranks (plumbing only)
    total_ms, e2e_lean_ms, e2e_full_ms, warm_ms, e2e_ov_ms = shard.max_over_ranks(
        [total_ms, e2e["lean"][0], e2e["full"][0], warm_ms, e2e_ov_ms], device=dev)
    ms_per_step = total_ms / args.steps
    value = shard.job_throughput(n_events, world, ms_per_step)

    # ---- roofline of the one kernel (per launch, this rank)
    hbm_gbs, hbm_src = hbm_peak()
    t_kernel = ms_per_step * 1e-3
    roof = roofline_block(wb, t_kernel, v_in, v_in_how, atom_rate, hbm_gbs, hbm_src, counts=alg_counts, atom_src=atom_src)
    # diagnostic third ceiling: the voting loop's own instruction sequence, alone on the SMs, measured now
    roof["vote_loop_probe"] = {"lane_votes_per_s_incl_padding": probe, "unit": "hit x theta pairs/s, 192 padded columns per 180",
                               "kernel_vs_probe": (wb.pairs * 192.0 / 180.0 / t_kernel) / probe if probe and w.n_theta == 180 else None,
                               "probe_vs_atomic_peak": probe / atom_rate if probe else None, "error": probe_err}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": workload_config(w, n_events, world, extra={
            "l2": "cold: 256 MiB write between steps" if flush is not None else "warm",
            "hits_per_gpu": n_total, "launch": info, "ms_per_step_warm_l2_back_to_back": warm_ms,
            "ms_per_step_min": float(times.min()), "ms_per_step_median": float(np.median(times)),
            "kept_fraction": alg_counts[0] / max(1, n_total), "quality": quality, "wall_s_timed_region": t_wall}),
        "gvotes_per_s": world * wb.pairs / t_kernel / 1e9,
        "gvotes_in_range_per_s": world * v_in / t_kernel / 1e9,
        "roofline": roof, "clocks": clocks,
        "e2e": {"value": None if "lean" in e2e_err else shard.job_throughput(n_events, world, e2e_lean_ms / e2e_steps), "unit": UNIT,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": e2e["lean"][1],
                "ms_per_step": None if "lean" in e2e_err else e2e_lean_ms / e2e_steps, "steps": e2e_steps, "error": e2e_err.get("lean"),
                "returns": "keep mask + peaks + counts (lean mode of hough_run_host)",
                "full": {"value": None if "full" in e2e_err else shard.job_throughput(n_events, world, e2e_full_ms / e2e_steps),
                         "d2h_bytes_per_step": e2e["full"][1], "ms_per_step": None if "full" in e2e_err else e2e_full_ms / e2e_steps,
                         "error": e2e_err.get("full"), "returns": "lean + kept_xy + kept_idx (full-length arrays)"},
                "overlapped_4_streams": {"value": None if e2e_ov_err else shard.job_throughput(n_events, world, e2e_ov_ms / e2e_steps),
                                         "ms_per_step": None if e2e_ov_err else e2e_ov_ms / e2e_steps, "error": e2e_ov_err,
                                         "what": "the lean transfer as 4 sub-batches on 4 streams, one staging area per stream (PAPER.md:228)"}},
        "gpu_launches": int(launches),
    }
    wb.close()

    # ---- every configuration of BASELINE.json in the same line (rank 0, single GPU; north_star: "events/s reported for every config")
    if rank == 0 and world == 1 and not args.no_all_configs and not args.vote_path:
        allc = []
        for cfg, nev, cl in ((0, 16, 0), (1, 1000, 0), (2, 1000, 0), (3, 1000, 0), (4, args.sweep_events, 0), (5, args.sweep_events, 0)):
            try:       # a configuration that fails is reported as such; it must not cost the headline line
                b2 = Workbench(hb, si, torch, dev, cfg, nev, staging=args.staging, scheduler=args.scheduler, select=args.select)
                fl = flush if b2.n_total * 8 < (96 << 20) else None       # inputs larger than L2 need no flush
                steps2 = args.config_steps if nev <= 1000 else max(5, args.config_steps // 4)
                t2 = b2.timed(steps2, 3, fl, stream)
                v2, how2 = b2.in_range_votes(None if nev <= 1000 else 2000)
                c = config_line(b2, t2, v2, how2, atom_rate, hbm_gbs, hbm_src)
                c["l2"] = "cold: 256 MiB write between steps" if fl is not None else "inputs (%d MB) exceed L2" % (b2.n_total * 8 >> 20)
                allc.append(c)
                if cfg == 4:
                    line["multi_stream"] = {"workload": b2.w.name, "events": nev,
                                            "what": "whole sweep in batches on 1/2/4 streams through one handle",
                                            "runs": multi_stream_sweep(b2, torch)}
                b2.close()
                del b2
            except Exception as ex:  # noqa: BLE001
                allc.append({"workload": si.config(cfg).name, "events": nev, "error": "%s: %s" % (type(ex).__name__, ex)})
            torch.cuda.empty_cache()
        line["all_configs"] = allc

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = len(os.sched_getaffinity(0))
        r1, dt1 = oracle_rate(w, xy, off, n_events, cores, 1)
        reps = max(1, min(50, int(12.0 / max(1e-3, dt1))))
        rN, dtN = oracle_rate(w, xy, off, n_events, cores, reps)
        rS, dtS = oracle_rate(w, xy, off, min(n_events, 250), 1, 1)
        line["cpu_baseline"] = {"value": rN, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "the whole %d-event batch x %d passes, %d threads (%.1f s wall); single thread on the first %d events: %.0f events/s"
                                          % (n_events, reps, cores, dtN, min(n_events, 250), rS),
                                "single_thread_value": rS}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.segment == "probes":
        return run_probe_segment()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
