"""bench.py's reference arm (the oracle on the host cores) prints the contract's JSON line; runs without a GPU."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "3",
                        "--warmup", "3", "--workload", "2"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "grid-point-steps/s" and line["higher_is_better"] is True
    assert line["value"] > 0 and line["steps"] == 3 and line["n_gpus"] == 1 and line["vs_baseline"] is None
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in line["config"] and line["gpu_launches"] == 0


def test_default_workload_is_the_metric_config():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.WORKLOADS["4"] == dict(cfg=4, dtype="c128")
    assert bench.METRIC.startswith("split-step")


def test_sweep_rejects_sizes_outside_the_supported_line_lengths():
    """--sweep (the paper's Figure 2: step time against N = 2^eta) takes 12 <= eta <= 26 only; the
    argument check runs before any GPU work."""
    for extra in (["--eta-max", "27"], ["--eta-min", "11"], ["--eta-min", "20", "--eta-max", "19"]):
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--sweep"] + extra, capture_output=True,
                           text=True, timeout=300, cwd=ROOT)
        assert r.returncode == 2 and "eta" in r.stderr
