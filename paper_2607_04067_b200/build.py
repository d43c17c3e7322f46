"""Builds paper_2607_04067_b200/libhough_b200.so for sm_100a with nvcc (in-tree;
nvcc cross-compiles without a GPU).  The kernels use __fmul_rn/__fadd_rn/__fadd_rd
and -fmad=false so that no multiply-add is ever contracted (S2); as a
belt-and-braces check the SASS must contain no packed FFMA2 and must contain the
floor-add (FADD.RM), the clamp (VIMNMX) and the vote (ATOMS.POPC.INC)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhough_b200.so")
SOURCES = ["hough_api.cu", "microbench.cu"]
HEADERS = ["hough_kernel.cuh", os.path.join("..", "..", "include", "hough.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
    "-shared", "-Xcompiler", "-fPIC", "-cudart", "static",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def check_sass(lib: str = LIB) -> None:
    sass = subprocess.run(["cuobjdump", "-sass", lib], check=True, capture_output=True, text=True).stdout
    if "FFMA2" in sass:
        raise RuntimeError("ptxas contracted a packed fp32 multiply-add (FFMA2 found): bit-exactness is lost")
    for needle in ("FADD.RM", "ATOMS.POPC.INC", "VIMNMX"):
        if needle not in sass:
            raise RuntimeError("expected %s in the SASS of %s" % (needle, lib))


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc, *NVCC_FLAGS] + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    check_sass(tmp)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
