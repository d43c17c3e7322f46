"""bench.py's reference arm (the oracle on the host cores) runs without a GPU and prints the contract's JSON line;
the argument parser and the helpers of the GPU arm are importable on a CPU box."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*argv, env=None):
    e = dict(os.environ)
    e.update(env or {})
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], capture_output=True, text=True, env=e, timeout=600)
    return r


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    r = run_bench("--impl", "reference", "--config", "0", "--steps", "2", "--warmup", "1")
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "events/s" and d["higher_is_better"] is True
    for k in ("metric", "value", "n_gpus", "steps", "warmup", "ms_per_step", "scaling", "vs_baseline", "dtype", "data", "config",
              "cpu_baseline", "e2e"):
        assert k in d, k
    assert d["vs_baseline"] is None and d["data"] == "synthetic" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and "model" not in d["config"]


def test_reference_arm_under_torchrun_env_only_rank0_prints():
    r = run_bench("--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "0", "--gpus", "2",
                  env={"RANK": "1", "LOCAL_RANK": "1", "WORLD_SIZE": "2"})
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_gpu_arm_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        import pytest
        pytest.skip("a GPU is present")
    r = run_bench("--steps", "1", "--warmup", "0")
    assert r.returncode != 0
    assert "no CPU fallback" in (r.stderr + r.stdout)


def test_default_arguments_and_blocks_of_the_gpu_arm():
    sys.path.insert(0, ROOT)
    import bench
    old = sys.argv
    try:
        sys.argv = ["bench.py"]
        a = bench.parse_args()
    finally:
        sys.argv = old
    assert a.gpus == 1 and a.config == 1 and a.warmup >= 3 and a.impl == "ours" and a.config_steps >= 20
    assert not a.no_all_configs and a.sweep_events == 100000
    src = open(os.path.join(ROOT, "bench.py")).read()
    for key in ('"roofline"', '"cpu_baseline"', '"e2e"', '"all_configs"', '"multi_stream"', '"gpu_launches"', '"clocks"'):
        assert key in src, key
    assert "_work" not in src and "/root/reference" not in src


def test_probe_segment_failure_falls_back_to_the_derived_peak_and_says_so():
    """The roofline denominator is measured in a child process; when that fails (here: no GPU) the line still carries a
    peak -- the derived 32 atomics per clock per SM -- and its source says it was not measured."""
    import torch
    if torch.cuda.is_available():
        import pytest
        pytest.skip("a GPU is present")
    sys.path.insert(0, ROOT)
    import bench
    rate, src, probe, probe_err = bench.device_probes(148, 1965, timeout_s=600)
    assert rate == 32.0 * 148 * 1965e6
    assert src.startswith("DERIVED, not measured") and probe is None and probe_err
