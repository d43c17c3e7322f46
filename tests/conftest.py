import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# HOUGH_GPU_TESTS_ON_EMULATOR=1: a DRY RUN of the gpu-marked tests on a box without a GPU, through the real Python binding
# and the real host code, kernels executed by the SIMT emulator at reduced event counts (tests/simt_emu/torch_shim.py).
# It checks the test files and the binding; it is not a parity claim and never on by default.  These need the real thing:
REAL_GPU_ONLY = ("test_cuda_graph_capture_and_replay", "test_second_device_when_present", "test_measurement_aids_run",
                 "test_shared_atomic_microbench_runs", "test_marshalling_rejects_wrong_dtype_device_and_length",
                 "test_cfg4_sweep_sampled_parity_100k",       # samples events of the whole 100k-event sweep
                 "test_work_stealing_scheduler_with_empty_refused_and_chunked_events_and_on_streams")   # indexes a 600-event batch
EMULATED = os.environ.get("HOUGH_GPU_TESTS_ON_EMULATOR") == "1"


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    if EMULATED:
        import torch
        if torch.cuda.is_available():
            raise pytest.UsageError("HOUGH_GPU_TESTS_ON_EMULATOR=1 on a box with a GPU: run the real tests")
        sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
        from simt_emu import torch_shim
        torch_shim.install()


def pytest_collection_modifyitems(config, items):
    # A gpu-marked test never silently passes on a box without a GPU.
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if EMULATED:
        skip = pytest.mark.skip(reason="needs a real GPU (dry run on the emulator)")
        for item in items:
            if "gpu" in item.keywords and item.originalname in REAL_GPU_ONLY:
                item.add_marker(skip)
        return
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device here; run with gpurun")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_collection_finish(session):
    """The emulator flavours the selected tests will ask for, compiled side by side up front (one g++ each; built one
    after the other they cost a minute and a half of a fresh checkout's first run)."""
    wanted = set()
    for item in session.items:
        mod = os.path.basename(str(item.fspath))
        if mod in ("test_kernel_emulation.py", "test_gpu_scenarios_under_emulator.py"):
            wanted.update(["emu", "emu_dbg"])
        elif mod == "test_kernel_races.py":
            wanted.add("emu_race")
        elif mod == "test_host_emulation.py":
            wanted.update(["host", "host_race"])
    if not wanted or session.config.option.collectonly:
        return
    from concurrent.futures import ThreadPoolExecutor
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    import simt_emu
    from simt_emu import host
    jobs = {"emu": lambda: simt_emu._build_locked(False, False, False), "emu_dbg": lambda: simt_emu._build_locked(True, False, False),
            "emu_race": lambda: simt_emu._build_locked(False, False, True), "host": lambda: host._build_unlocked(False),
            "host_race": lambda: host._build_unlocked(True)}
    try:
        with ThreadPoolExecutor(len(wanted)) as ex:
            list(ex.map(lambda k: jobs[k](), sorted(wanted)))
    except Exception:  # noqa: BLE001 -- the test that needs the build reports the failure
        pass
