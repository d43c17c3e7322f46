"""Builds the native libraries for sm_100a with nvcc, in-tree (nvcc cross-compiles without a GPU):

  libhough_b200.so      the product: C ABI of include/hough.h (+ the host-only introspection of include/hough_debug.h)
  libhough_b200_dbg.so  the same sources with -DHOUGH_DEBUG_BOUNDS: every shared-memory offset of the kernel is checked
                        before use, a violating access is skipped and reported in d_counts (never traps); the first
                        thing to run on a GPU after any change of the kernel's addressing (HOUGH_B200_FLAVOR=dbg)
  libhough_b200_diag.so bench-only: -DHOUGH_DIAG adds the phase-skipping timing diagnostics (HOUGH_B200_FLAVOR=diag)
  libhough_bench.so     measurement aids of include/hough_bench.h (roofline denominator, instruction-cost probes)

The kernels use __fmul_rn/__fadd_rn/__fadd_rd and -fmad=false so that no multiply-add is ever contracted (DESIGN.md
S2); as a belt-and-braces check the product's SASS must contain no packed FFMA2 and must contain the floor-add
(FADD.RM), the clamp (VIMNMX) and the vote (ATOMS.POPC.INC); the bulk-copy staging option must show up as UBLKCP, the work-stealing
scheduler as UGETNEXTWORKID (cluster launch control) and UBLKPF (L2 prefetch), and only in the extended instantiations."""
import os
import re
import subprocess
import sys
import threading

_BUILD_LOCK = threading.Lock()      # one build at a time per process (the temporary file is named after the pid)

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(HERE, "..", "include")
HEADERS = [os.path.join(CSRC, "hough_kernel.cuh"), os.path.join(INCLUDE, "hough.h"), os.path.join(INCLUDE, "hough_debug.h"),
           os.path.join(INCLUDE, "hough_bench.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
    "-shared", "-Xcompiler", "-fPIC", "-cudart", "static",
]
FLAVORS = {
    "release": ("libhough_b200.so", ["hough_api.cu"], []),
    "dbg": ("libhough_b200_dbg.so", ["hough_api.cu"], ["-DHOUGH_DEBUG_BOUNDS"]),
    "diag": ("libhough_b200_diag.so", ["hough_api.cu"], ["-DHOUGH_DIAG"]),
    "bench": ("libhough_bench.so", ["microbench.cu"], []),
}
LIB = os.path.join(HERE, FLAVORS["release"][0])
BENCH_LIB = os.path.join(HERE, FLAVORS["bench"][0])


def lib_path(flavor: str = "release") -> str:
    return os.path.join(HERE, FLAVORS[flavor][0])


def _stale(flavor: str) -> bool:
    lib = lib_path(flavor)
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in FLAVORS[flavor][1]] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _sass(lib: str) -> str:
    return subprocess.run(["cuobjdump", "-sass", lib], check=True, capture_output=True, text=True).stdout


def check_sass(lib: str = LIB) -> None:
    sass = _sass(lib)
    if "FFMA2" in sass:
        raise RuntimeError("ptxas contracted a packed fp32 multiply-add (FFMA2 found): bit-exactness is lost")
    for needle in ("FADD.RM", "ATOMS.POPC.INC", "VIMNMX", "UBLKCP", "UGETNEXTWORKID", "UBLKPF"):
        if needle not in sass:
            raise RuntimeError("expected %s in the SASS of %s" % (needle, lib))
    # the default instantiations (EXT = false, last template argument Lb0E) carry none of the optional paths:
    # no bulk copy / mbarrier / launch control, no fp64 arithmetic of the distance filter
    for m in re.finditer(r"Function : (\S*hough_event_kernelI\S*ELb0EEE\S*)\n(.*?)(?=\n\s*Function : |\Z)", sass, flags=re.S):
        for needle in ("UBLKCP", "UBLKPF", "UGETNEXTWORKID", "SYNCS", "DADD", "DMUL", "DFMA"):
            if needle in m.group(2):
                raise RuntimeError("%s found in the default instantiation %s" % (needle, m.group(1)))


# hough_bench_issue_rate(kind): SASS opcodes that one loop trip of issue_kernel<kind> must hold, and how many
ISSUE_KINDS = {
    0: {"FMUL": 32}, 1: {"FADD": 32}, 2: {"FFMA": 32}, 3: {"FMUL2": 32}, 4: {"FADD2": 32}, 5: {"IMAD": 32},
    6: {"VIMNMX": 32}, 7: {"IADD3": 32}, 8: {"LOP3": 32}, 9: {"LEA": 32},
    10: {"FMUL": 16, "VIMNMX": 16}, 11: {"FMUL": 16, "IMAD": 16}, 12: {"FMUL2": 16, "VIMNMX": 16}, 13: {"FMUL": 16, "IADD3": 16},
}


def issue_kernel_loop_census(lib: str = BENCH_LIB) -> dict:
    """{kind: {opcode: count}} of the instructions inside the timed loop of every issue_kernel<kind> (between the
    loop head and the backward branch).  Used by check_bench_sass() and quoted in profiles/."""
    sass = _sass(lib)
    out = {}
    for m in re.finditer(r"Function : (\S*issue_kernelILi(\d+)E\S*)\n(.*?)(?=\n\s*Function : |\Z)", sass, flags=re.S):
        kind, body = int(m.group(2)), m.group(3)
        lines = [l for l in body.splitlines() if re.search(r"/\*[0-9a-f]{4}\*/", l)]
        addr = lambda l: int(re.search(r"/\*([0-9a-f]{4})\*/", l).group(1), 16)
        # the backward branch with the longest span closes the (unrolled) timed loop
        loop = None
        for i, l in enumerate(lines):
            b = re.search(r"\bBRA\b.*?0x([0-9a-f]+)", l)
            if b and int(b.group(1), 16) < addr(l) and (loop is None or addr(l) - int(b.group(1), 16) > loop[1] - loop[0]):
                loop = (int(b.group(1), 16), addr(l))
        census = {}
        if loop:
            for l in lines:
                if loop[0] <= addr(l) <= loop[1]:
                    op = re.search(r"\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)", l)
                    if op:
                        census[op.group(1)] = census.get(op.group(1), 0) + 1
        out[kind] = census
    return out


def check_bench_sass(lib: str = BENCH_LIB) -> dict:
    census = issue_kernel_loop_census(lib)
    for kind, want in ISSUE_KINDS.items():
        got = census.get(kind, {})
        for op, n in want.items():
            # ptxas balances the integer pipes itself: about half of a run of plain adds (and of shift-adds) is
            # emitted as IMAD (x*1+y, x*128+y) on the FMA pipe, the rest as IADD3 / LEA on the ALU pipe.  Count the family.
            fam = {"IADD3": ("IADD3", "IADD", "IMAD"), "LEA": ("LEA", "IMAD")}.get(op, (op,))
            have = sum(c for o, c in got.items() if o in fam)
            if have % n != 0 or have == 0:
                raise RuntimeError("issue_kernel<%d>: expected a multiple of %d %s in the loop, found %s" % (kind, n, op, got))
    return census


def build(flavor: str = "release", force: bool = False, verbose: bool = False) -> str:
    with _BUILD_LOCK:
        return _build_locked(flavor, force, verbose)


def _build_locked(flavor: str, force: bool, verbose: bool) -> str:
    lib = lib_path(flavor)
    if not force and not _stale(flavor):
        return lib
    name, sources, defs = FLAVORS[flavor]
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = lib + ".tmp.%d" % os.getpid()
    cmd = [nvcc, *NVCC_FLAGS, *defs] + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, s) for s in sources]
    subprocess.check_call(cmd)
    if flavor == "bench":
        check_bench_sass(tmp)
    else:
        check_sass(tmp)
    os.replace(tmp, lib)
    return lib


def build_all(force: bool = False, verbose: bool = False):
    return [build(f, force=force, verbose=verbose) for f in ("release", "dbg", "bench")]


if __name__ == "__main__":
    flavors = [a for a in sys.argv[1:] if a in FLAVORS] or ["release", "dbg", "bench"]
    for f in flavors:
        print(build(f, force=True, verbose="-v" in sys.argv))
