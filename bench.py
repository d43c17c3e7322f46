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
                        buffers: H2D of hits+offsets and D2H of mask, peaks,
                        counts and the compacted hits inside the timed region
  roofline            : achieved in-range votes/s of the one kernel against the
                        shared-atomic rate measured live on this GPU, plus the
                        HBM term (north_star: the slower of the two binds)
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
    ap.add_argument("--vote-path", type=int, default=0, help="HOUGH_OPT_VOTE_PATH (0 packed fast, 1 exact slow)")
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


def dram_traffic(workload_name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernel, from the committed ncu capture
    (profiles/dram_traffic.csv); None when this workload has no capture."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "dram_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload_name:
                    return int(row["dram_bytes_read_per_launch"]) + int(row["dram_bytes_write_per_launch"])
    except Exception:  # noqa: BLE001
        pass
    return None


def run_ours(args):
    import numpy as np
    import torch
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
    xy, off, _ = si.generate(w, n_events, first_event=first_event)
    n_total = len(xy)
    table = si.trig_table(w.n_theta)
    h = hb.Hough(w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, max_peaks=w.max_peaks, acc_dtype=w.acc_dtype,
                 cluster_size=args.cluster, ctas_per_sm=args.ctas_per_sm, trig_table=table)
    if args.vote_path:
        hb.hough_set_option(h.ctx, hb.HOUGH_OPT_VOTE_PATH, args.vote_path)
    info = {k: h.info(getattr(hb, "HOUGH_INFO_" + k)) for k in
            ("CLUSTER_SIZE", "THREADS", "SMEM_BYTES", "CTAS_PER_SM", "GRID_MAX", "ACC_BITS", "CHUNK_HITS", "SM_COUNT")}
    info["VOTE_PATH"] = args.vote_path
    d_xy = torch.from_numpy(xy).to(dev)
    d_off = torch.from_numpy(off).to(dev)
    out = h.alloc_outputs(n_total, n_events, dev, kept=True, accum=False)
    stream = torch.cuda.current_stream()

    pairs = n_total * w.n_theta
    flush = None if args.no_flush else torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step():
        hb.hough_run_ex(h.ctx, d_xy, d_off, n_events, out["keep"], out["peaks"], out["counts"],
                        out["kept_xy"], out["kept_idx"], None, stream)

    for _ in range(max(args.warmup, 3)):
        if flush is not None:
            flush.zero_()
        step()
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
        step()
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
        step()
    b.record(stream)
    torch.cuda.synchronize()
    warm_ms = a.elapsed_time(b) / args.steps

    # ---- end to end through hough_run_host: pinned host buffers, copies inside the timed region
    h_xy, h_off = torch.from_numpy(xy).pin_memory(), torch.from_numpy(off).pin_memory()
    h_keep = torch.empty(n_total, dtype=torch.uint8).pin_memory()
    h_peaks = torch.zeros((n_events, w.max_peaks, 2), dtype=torch.int32).pin_memory()
    h_counts = torch.empty((n_events, 2), dtype=torch.int32).pin_memory()
    h_kxy = torch.empty((n_total, 2), dtype=torch.float32).pin_memory()
    h_kidx = torch.empty(n_total, dtype=torch.int32).pin_memory()
    e2e_steps = min(args.steps, 50)
    for _ in range(3):
        hb.hough_run_host(h.ctx, h_xy, h_off, n_events, h_keep, h_peaks, h_counts, h_kxy, h_kidx, stream)
    torch.cuda.synchronize()
    barrier()
    e2e_ms = 0.0
    for _ in range(e2e_steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        hb.hough_run_host(h.ctx, h_xy, h_off, n_events, h_keep, h_peaks, h_counts, h_kxy, h_kidx, stream)
        b.record(stream)
        b.synchronize()               # the caller reads the results on the host here
        e2e_ms += a.elapsed_time(b)
    barrier()
    n_kept = int(h_counts[:, 1].sum().item())
    n_peaks = int(h_counts[:, 0].clamp(max=w.max_peaks).sum().item())
    h2d = h_xy.numel() * 4 + h_off.numel() * 4
    d2h = h_keep.numel() + h_peaks.numel() * 4 + h_counts.numel() * 4 + h_kxy.numel() * 4 + h_kidx.numel() * 4

    # in-range votes V_in = sum of all accumulator cells (the roofline's unit), from the kernel's own dump;
    # untimed, and after the timed regions so that a profiler's first hough launches are the real ones
    v_in = 0
    step_ev = 125
    for e0 in range(0, n_events, step_ev):
        e1 = min(n_events, e0 + step_ev)
        sub_off = (d_off[e0:e1 + 1] - d_off[e0]).contiguous()
        sub_xy = d_xy[int(off[e0]):int(off[e1])]
        o = h.run(sub_xy, sub_off, kept=False, accum=True)
        v_in += int(o["accum"].sum(dtype=torch.int64).item())
        del o


    # ---- max over ranks (plumbing only)
    total_ms, e2e_ms, warm_ms = shard.max_over_ranks([total_ms, e2e_ms, warm_ms], device=dev)
    ms_per_step = total_ms / args.steps
    value = shard.job_throughput(n_events, world, ms_per_step)
    e2e_value = shard.job_throughput(n_events, world, e2e_ms / e2e_steps)

    # ---- roofline of the one kernel (per launch, this rank)
    atom_rate = hb.hough_bench_shared_atomics(5, 1, 1024, 20000)          # conflict-free ATOMS/s, all SMs, measured now
    hbm_gbs, hbm_src = hbm_peak()
    alg_bytes = 8 * n_total + 4 * (n_events + 1) + n_total + 12 * n_kept + 8 * n_peaks + 8 * n_events
    t_kernel = ms_per_step * 1e-3
    t_vote, t_hbm = v_in / atom_rate, alg_bytes / (hbm_gbs * 1e9)
    roof = {
        "bound": "alu", "pipe": "shared-memory atomics (ATOMS), one per in-range vote; the slower of the vote and HBM terms binds (north_star)",
        "achieved": v_in / t_kernel / 1e9, "peak": atom_rate / 1e9, "unit": "Gvotes/s (in-range)",
        "frac": max(t_vote, t_hbm) / t_kernel, "traffic": dram_traffic(w.name),
        "peak_source": "hough_bench_shared_atomics(variant 5) measured in this run: conflict-free 32-bit shared atomics, all SMs",
        "algorithmic_votes_per_launch": v_in, "algorithmic_bytes_per_launch": alg_bytes,
        "t_vote_us": t_vote * 1e6, "t_hbm_us": t_hbm * 1e6, "t_kernel_us": t_kernel * 1e6,
        # diagnostic third ceiling: 10.3 issue slots per (hit, theta) vote, 4 slots per clock per SM
        "issue_slot_ceiling": {"slots_per_vote": 10.3, "peak": info["SM_COUNT"] * (clocks.get("sm_mhz") or 1965) * 1e6 * 128 / 10.3 / 1e9,
                               "achieved": pairs / t_kernel / 1e9, "unit": "Gvotes/s (hit x theta)",
                               "frac": (pairs / t_kernel) / (info["SM_COUNT"] * (clocks.get("sm_mhz") or 1965) * 1e6 * 128 / 10.3),
                               "source": "profiles/r01_microbench_voteloop.md"},
        "hbm": {"achieved": alg_bytes / t_kernel / 1e9, "peak": hbm_gbs, "unit": "GB/s", "frac": t_hbm / t_kernel, "peak_source": hbm_src},
    }

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": workload_config(w, n_events, world, extra={
            "l2": "cold: 256 MiB write between steps" if flush is not None else "warm",
            "hits_per_gpu": n_total, "launch": info, "ms_per_step_warm_l2_back_to_back": warm_ms,
            "ms_per_step_min": float(times.min()), "ms_per_step_median": float(np.median(times)),
            "kept_fraction": n_kept / max(1, n_total), "wall_s_timed_region": t_wall}),
        "gvotes_per_s": world * pairs / t_kernel / 1e9,
        "gvotes_in_range_per_s": world * v_in / t_kernel / 1e9,
        "roofline": roof, "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps},
        "gpu_launches": int(launches),
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = len(os.sched_getaffinity(0))
        r1, dt1 = oracle_rate(w, xy, off, n_events, cores, 1)
        reps = max(1, min(50, int(12.0 / max(1e-3, dt1 * cores))))
        rN, dtN = oracle_rate(w, xy, off, n_events, cores, reps)
        rS, dtS = oracle_rate(w, xy, off, min(n_events, 250), 1, 1)
        line["cpu_baseline"] = {"value": rN, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "the whole %d-event batch x %d passes, %d threads (%.1f s wall); single thread on the first %d events: %.0f events/s"
                                          % (n_events, reps, cores, dtN, min(n_events, 250), rS),
                                "single_thread_value": rS}
    h.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
