"""bench.py --impl reference on the CPU: the oracle arm of the bench contract prints one JSON line with the
contract's keys for an SMC workload and for a nested-sampling workload (no GPU, no CUDA library)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KEYS = {"impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
        "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"}


def run(*extra):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", *extra], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    return json.loads(out.stdout.strip().splitlines()[-1])


def test_reference_arm_smc_small_workload():
    d = run("--workload", "C0")
    assert KEYS <= set(d) and d["impl"] == "reference" and d["metric"] == "site-updates/s"
    assert d["value"] > 0 and d["gpu_launches"] == 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"].startswith("C0")


def test_reference_arm_nested_sampling_workload():
    d = run("--workload", "C2")
    assert KEYS <= set(d) and d["impl"] == "reference" and d["value"] > 0
    assert d["config"]["n_live"] == 4096 and d["config"]["k_delete"] == 512
    assert d["config"]["iterations_per_step"] == [64]          # a bounded sample of the run
