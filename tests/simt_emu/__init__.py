"""TEST INFRASTRUCTURE: runs the CUDA kernel's source (paper_2607_04067_b200/csrc/hough_kernel.cuh) on the CPU under a
small SIMT emulator (simt_shim.h: fibers, barriers, warp collectives, guarded shared memory), so that the `-m "not
gpu"` tests can compare the kernel's LOGIC with the oracle without a GPU.  Not a product path and not a parity claim:
the product library never loads this, and only the GPU tests say anything about the device code itself.

The launch shape and the shared-memory layout are asked from the product's own planner (hough_plan_describe), the
tame bounds from hough_debug_tame_bounds, so the emulated launch is the one hough_run would make."""
import os
import struct
import subprocess
import tempfile
import threading

import numpy as np

# the layout of hough_circle (include/hough.h)
CIRCLE_DTYPE = np.dtype([("x_c", "<f8"), ("y_c", "<f8"), ("r_c", "<f8"), ("pt", "<f8"), ("phi0", "<f8"), ("charge", "<i4"), ("n_hits", "<i4")])

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
SOURCES = [os.path.join(HERE, "emu_main.cpp"), os.path.join(HERE, "simt_shim.h"),
           os.path.join(ROOT, "paper_2607_04067_b200", "csrc", "hough_kernel.cuh"), os.path.join(ROOT, "include", "hough.h"),
           os.path.abspath(__file__)]
FLAGS = ["-O1", "-g", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-DHOUGH_HOST_EMU", "-Wno-unused-variable"]


def exe_path(debug_bounds: bool, race: bool = False) -> str:
    return os.path.join(HERE, "hough_emu_race" if race else "hough_emu_dbg" if debug_bounds else "hough_emu")


def _compile(exe: str, extra, race: bool) -> None:
    if not race:
        subprocess.check_call(["g++", *FLAGS, *extra, "-o", exe, SOURCES[0]])
        return
    # the race-check build: the compiler's -fsanitize=thread instrumentation, linked WITHOUT ThreadSanitizer's runtime
    # (the hooks are in simt_shim.h); no PIE, so that the reported code addresses can be looked up with addr2line
    obj = exe + ".o"
    subprocess.check_call(["g++", *FLAGS, *extra, "-fsanitize=thread", "-no-pie", "-c", "-o", obj, SOURCES[0]])
    subprocess.check_call(["g++", "-no-pie", "-o", exe, obj])
    os.remove(obj)


_BUILD_LOCK = threading.Lock()


def build(debug_bounds: bool = False, force: bool = False, race: bool = False) -> str:
    with _BUILD_LOCK:
        return _build_locked(debug_bounds, force, race)


def _build_locked(debug_bounds: bool, force: bool, race: bool) -> str:
    exe = exe_path(debug_bounds, race)
    if not force and os.path.exists(exe) and all(os.path.getmtime(s) <= os.path.getmtime(exe) for s in SOURCES):
        return exe
    tmp = exe + ".tmp.%d" % os.getpid()
    _compile(tmp, ["-DHOUGH_DEBUG_BOUNDS"] if debug_bounds and not race else [], race)
    os.replace(tmp, exe)
    return exe


def build_mutant(exe: str, edits, race: bool = True) -> str:
    """Compiles the emulator against a COPY of the kernel source with `edits` = [(old, new), ...] applied (each `old`
    must occur exactly once) and writes it to `exe`: the mutation tests of the race check."""
    src = open(SOURCES[2]).read()
    for old, new in edits:
        if src.count(old) != 1:
            raise ValueError("mutation anchor occurs %d times: %r" % (src.count(old), old))
        src = src.replace(old, new)
    src = src.replace('"../../include/hough.h"', '"%s"' % SOURCES[3])
    hdr = exe + ".cuh"
    with open(hdr, "w") as f:
        f.write(src)
    _compile(exe, ['-DHOUGH_KERNEL_HEADER="%s"' % hdr], race)
    return exe


class RaceReport(RuntimeError):
    """The race-check build found conflicting accesses that no barrier orders.  .reports: one dict per distinct pair of
    code locations: {"text": the emulator's line, "now": "function file:line", "earlier": "function file:line"}."""

    def __init__(self, reports):
        self.reports = reports
        super().__init__("%d race report(s):\n%s" % (len(reports), "\n".join(
            "%s\n    now:     %s\n    earlier: %s" % (r["text"], r["now"], r["earlier"]) for r in reports[:6])))


def _symbolize(exe: str, pcs):
    """{pc: "function file:line <- inlined into file:line <- ..."} (addr2line -i: the whole inline chain, innermost first)."""
    out = subprocess.run(["addr2line", "-e", exe, "-a", "-f", "-C", "-s", "-i", *pcs], capture_output=True, text=True).stdout.splitlines()
    sym, key, frames = {}, None, []
    for l in out + ["0x"]:
        if l.startswith("0x"):
            if key is not None:
                sym[key] = " <- ".join("%s %s" % (frames[i][:50], frames[i + 1]) for i in range(0, len(frames) - 1, 2)) or "?"
            key, frames = "0x%x" % int(l, 16) if len(l) > 2 else None, []
        else:
            frames.append(l)
    return sym


def _race_reports(exe: str, stderr: str):
    import re
    lines = [l for l in stderr.splitlines() if l.startswith("RACE ") or l.startswith("UNINIT ")]
    pcs = sorted({pc for l in lines for pc in re.findall(r"pc (0x[0-9a-f]+)", l)})
    sym = _symbolize(exe, pcs) if pcs else {}
    reports = []
    for l in lines:
        found = re.findall(r"pc (0x[0-9a-f]+)", l)
        reports.append({"text": l, "now": sym.get(found[0], "?"), "earlier": sym.get(found[1], "?") if len(found) > 1 else "-"})
    return reports


def run(xy, off, n_theta, n_rho, rho_max, threshold, window, table, max_peaks=64, acc_dtype="u16", accum=True,
        conformal_scale=1, cluster_size=0, ctas_per_sm=0, vote_path=0, grid_clusters=0, debug_bounds=False, timeout=900,
        peak_mode=0, rel_permille=500, nms_radius=1, theta_wrap=False, keep_mode=0, keep_tol=0.0, b_field=1.0, circles=False,
        order=None, staging=0, scheduler=0, steals=None, race=False, exe=None, select_mode=0):
    """Same arguments and result keys as tests/test_parity_gpu.py::gpu_run."""
    import paper_2607_04067_b200 as hb
    xy = np.ascontiguousarray(xy, dtype=np.float32).reshape(-1, 2)
    off = np.ascontiguousarray(off, dtype=np.int32)
    n_events, n_total = len(off) - 1, len(xy)
    acc = {"auto": hb.HOUGH_ACC_AUTO, "u16": hb.HOUGH_ACC_U16, "u32": hb.HOUGH_ACC_U32}[acc_dtype]
    plan = hb.hough_plan_describe(n_theta, n_rho, acc, cluster_size=cluster_size, ctas_per_sm=ctas_per_sm)
    fields = [plan[k] for k in hb.PLAN_FIELDS]
    c, s = (np.ascontiguousarray(t, dtype=np.float32) for t in table)
    tab = np.concatenate([np.abs(c), np.abs(s)])
    nz = tab[tab > 0]
    rho_max32 = float(np.float32(rho_max))
    tame, ftz_min = hb.hough_debug_tame_bounds(n_rho, rho_max32, float(tab.max()), float(nz.min()) if nz.size else 0.0)
    inv = np.float32(float(n_rho) / (2.0 * rho_max32))
    head = [n_theta, n_rho, threshold, window, max_peaks, int(plan["acc_bits"] == 16), int(plan["cluster_size"] > 1),
            plan["cols_per_lane"], plan["cluster_size"], plan["threads"], plan["smem_bytes"], int(vote_path == 1),
            n_events, n_total, 1, int(accum), grid_clusters, peak_mode, rel_permille, nms_radius, int(bool(theta_wrap)), keep_mode,
            int(circles), int(staging) | (int(scheduler) << 1) | (int(select_mode) << 2)]
    with tempfile.TemporaryDirectory() as d:
        fin, fout = os.path.join(d, "in.bin"), os.path.join(d, "out.bin")
        with open(fin, "wb") as f:
            f.write(struct.pack("<24i", *head))
            f.write(struct.pack("<27i", *fields))
            f.write(struct.pack("<5f", rho_max32, float(inv), float(conformal_scale), tame, ftz_min))
            f.write(struct.pack("<2d", float(keep_tol), float(b_field)))
            f.write(c.tobytes()); f.write(s.tobytes()); f.write(off.tobytes()); f.write(xy.tobytes())
        env = dict(os.environ)
        if order:                      # fiber scheduling order: "reverse", "shuffle:<seed>" (simt_shim.h run_cluster)
            env["HOUGH_EMU_ORDER"] = order
        else:
            env.pop("HOUGH_EMU_ORDER", None)
        env.pop("HOUGH_EMU_STEALS", None)
        if steals is not None:         # launch control: events a CTA may take over before its requests fail (default: no limit)
            env["HOUGH_EMU_STEALS"] = str(int(steals))
        race = race or os.environ.get("HOUGH_EMU_RACE") == "1"     # HOUGH_EMU_RACE=1: every emulator test becomes a race check too
        exe = exe or build(debug_bounds, race=race)
        r = subprocess.run([exe, fin, fout], capture_output=True, text=True, timeout=timeout, env=env)
        if race and (r.returncode == 66 or r.stderr.startswith(("RACE ", "UNINIT "))):      # (a report may be followed by a crash)
            raise RaceReport(_race_reports(exe, r.stderr))
        if r.returncode != 0:
            raise RuntimeError("hough_emu failed (rc %d): %s" % (r.returncode, r.stderr.strip()[-400:]))
        raw = open(fout, "rb").read()
    o = 0
    def take(n, dtype):
        nonlocal o
        a = np.frombuffer(raw, dtype=dtype, count=n, offset=o)
        o += a.nbytes
        return a
    res = {"keep": take(n_total, np.uint8),
           "peaks": take(n_events * max_peaks * 2, np.int32).reshape(n_events, max_peaks, 2),
           "counts": take(2 * n_events, np.int32).reshape(n_events, 2),
           "kept_xy": take(2 * n_total, np.float32).reshape(n_total, 2),
           "kept_idx": take(n_total, np.int32)}
    if accum:
        res["accum"] = take(n_events * n_theta * n_rho, np.int32).reshape(n_events, n_theta, n_rho)
    if circles:
        res["circles"] = take(n_events * max_peaks, CIRCLE_DTYPE).reshape(n_events, max_peaks)
    if race and env.get("HOUGH_EMU_PROFILE"):       # {(file:line, "shared"|"global", kind): thread-level accesses}
        import re
        rows = [l.split() for l in r.stderr.splitlines() if l.startswith("PROF ")]
        sym = _symbolize(exe, sorted({x[2] for x in rows}))
        prof = {}
        for _, _, pc, space, kind, n in rows:
            m = re.search(r"(hough_kernel\.cuh:\d+)", sym.get(pc, ""))           # the kernel line of the inline chain
            key = (m.group(1) if m else sym.get(pc, pc), space, kind)
            prof[key] = prof.get(key, 0) + int(n)
        res["profile"] = prof
    res["peaks3"] = hb.unpack_peaks(res["peaks"])
    res["info"] = {"CLUSTER_SIZE": plan["cluster_size"], "THREADS": plan["threads"], "SMEM_BYTES": plan["smem_bytes"],
                   "ACC_BITS": plan["acc_bits"], "CHUNK_HITS": plan["chunk_hits"]}
    return res
