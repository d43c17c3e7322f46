"""-m "not gpu": the C-ABI library builds, loads and exports every symbol that
include/hough.h declares; without a GPU the product path fails loudly (no CPU
fallback)."""
import os
import re

import pytest

import paper_2607_04067_b200 as hb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions(header):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hough_[a-z_0-9]+)\s*\(", src)))


def test_libraries_export_every_symbol_the_headers_declare():
    # include/hough.h = the product ABI; hough_debug.h = host-only introspection of the same library;
    # hough_bench.h = measurement aids in their own library (never loaded by the product path)
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["hough.h", "hough_bench.h", "hough_debug.h"]
    lib = hb.load_library()
    assert set(declared_functions("hough.h")) == set(hb.EXPORTS)
    assert set(declared_functions("hough_debug.h")) == set(hb.DEBUG_EXPORTS)
    for n in hb.EXPORTS + hb.DEBUG_EXPORTS:
        assert hasattr(lib, n), n
    assert b"sm_100a" in lib.hough_version()
    bench = hb.load_bench_library()
    assert set(declared_functions("hough_bench.h")) == set(hb.BENCH_EXPORTS)
    for n in hb.BENCH_EXPORTS:
        assert hasattr(bench, n), n
        assert not hasattr(lib, n), "measurement aid %s leaked into the product library" % n


def test_debug_bounds_flavor_builds_and_says_so():
    import ctypes
    from paper_2607_04067_b200 import build
    dbg = ctypes.CDLL(build.build("dbg"))
    assert dbg.hough_debug_bounds_enabled() == 1 and not hb.hough_debug_bounds_enabled()
    dbg.hough_version.restype = ctypes.c_char_p
    assert b"debug bounds" in dbg.hough_version()
    for n in hb.EXPORTS + hb.DEBUG_EXPORTS:
        assert hasattr(dbg, n), n


def test_binding_mirrors_the_c_names():
    for n in hb.EXPORTS + hb.DEBUG_EXPORTS + hb.BENCH_EXPORTS:
        if n in ("hough_strerror", "hough_last_error"):
            continue
        assert callable(getattr(hb, n)), n


def test_strerror_and_status_codes():
    lib = hb.load_library()
    assert lib.hough_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4):
        assert lib.hough_strerror(code) not in (b"ok", b"unknown status")


def test_sass_has_floor_add_clamp_and_shared_atomics_and_no_contraction():
    from paper_2607_04067_b200 import build
    build.check_sass(hb.lib_path())    # raises if FFMA2 is present or FADD.RM / VIMNMX / ATOMS.POPC.INC are missing
    build.check_sass(build.build("dbg"))
    census = build.check_bench_sass(build.build("bench"))   # the instruction-rate probes hold the instructions they name
    assert census[0].get("FMUL", 0) % 32 == 0 and census[3].get("FMUL2", 0) % 32 == 0 and census[6].get("VIMNMX", 0) % 32 == 0


def test_no_gpu_means_loud_failure_not_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(hb.HoughError, match="no CUDA device|CUDA"):
        hb.hough_create(180, 256, 0.003, 16, 1)
    with pytest.raises(hb.HoughError):
        hb.hough_bench_shared_atomics(0, 1, 256, 10)
    with pytest.raises(hb.HoughError):
        hb.hough_bench_issue_rate(0, 1, 256, 10)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_04067_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "hough_oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2607_04067_b200\b", txt, flags=re.M), f
            assert "hough_kernel" not in txt and "libhough_b200" not in txt, f
