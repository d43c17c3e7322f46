"""TEST INFRASTRUCTURE: counts the kernel's shared- and global-memory operations per phase, thread by thread, by running
the kernel source under the emulator's race-check build with HOUGH_EMU_PROFILE=1 (simt_shim.h counts every instrumented
access of tracked memory per code address).  Not a timing and not a hardware counter: a statement of how much work each
phase does on a given workload, e.g. how many (hit, marked column) evaluations H6 makes against the (hit, column)
votes of H3.  Phases are the `// ----` section comments of hough_kernel.cuh.

    python tests/simt_emu/access_profile.py [--select MODE] [config events]...      (default: 1 8  2 4  3 3)

--select: HOUGH_OPT_SELECT_MODE of the run (0 scan, 1 dense, 2 auto).
"""
import os
import re
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))


def main(argv):
    select = 0
    if argv[:1] == ["--select"]:
        select, argv = int(argv[1]), argv[2:]
    os.environ["HOUGH_EMU_PROFILE"] = "1"
    import simt_emu
    import stcf_inputs as si
    src = open(simt_emu.SOURCES[2]).read().splitlines()
    marks = [(i + 1, l.strip()[8:66].strip(" -")) for i, l in enumerate(src) if l.strip().startswith("// ----")]

    def phase(line):
        cur = "set-up"
        for ln, name in marks:
            if ln <= line:
                cur = name or cur
        return cur
    pairs = [(int(argv[i]), int(argv[i + 1])) for i in range(0, len(argv) - 1, 2)] or [(1, 8), (2, 4), (3, 3)]
    for cfg, nev in pairs:
        w = si.config(cfg)
        xy, off, _ = si.generate(w, nev)
        r = simt_emu.run(xy, off, w.n_theta, w.n_rho, w.rho_max, w.threshold, w.window, si.trig_table(w.n_theta), max_peaks=w.max_peaks,
                         acc_dtype=w.acc_dtype, accum=False, race=True, select_mode=select)
        agg = {}
        for (loc, space, kind), n in r["profile"].items():
            m = re.search(r":(\d+)", loc)
            key = (phase(int(m.group(1))) if m else loc, space, kind)
            agg[key] = agg.get(key, 0) + n
        n_hits = len(xy)
        print("\n%s%s: %d events, %d hits, %d x %d %s, %d threads; stored peaks per event %.0f, kept fraction %.2f"
              % (w.name, " (select mode %d)" % select if select else "", nev, n_hits, w.n_theta, w.n_rho, w.acc_dtype, r["info"]["THREADS"], r["counts"][:, 0].clip(max=w.max_peaks).mean(),
                 r["counts"][:, 1].sum() / max(1, n_hits)))
        print("| phase | memory | access | thread-level operations | per hit |\n|---|---|---|---|---|")
        for k, n in sorted(agg.items(), key=lambda kv: -kv[1]):
            if n * 200 >= n_hits:
                print("| %s | %s | %s | %d | %.1f |" % (k[0], k[1], k[2], n, n / n_hits))


if __name__ == "__main__":
    main(sys.argv[1:])
