"""bench.py's reference arm runs anywhere (it times the CPU oracle): check the JSON contract of the line it prints,
and that the CUDA arm refuses to run without a device instead of falling back."""
import json
import os
import subprocess
import sys

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(*args):
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                          timeout=300, cwd=ROOT)


def test_reference_arm_prints_one_contract_line():
    r = run("--impl", "reference", "--workload", "c1", "--steps", "1", "--warmup", "0")
    assert r.returncode == 0, r.stderr
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["unit"] == "docs/s" and j["higher_is_better"] is True
    assert j["value"] > 0 and j["steps"] == 1 and j["n_gpus"] == 1 and j["dtype"] == "f64" and j["data"] == "synthetic"
    assert j["config"]["workload"].startswith("c1") and "model" not in j["config"]
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] >= 1
    assert j["e2e"] == {"value": j["value"], "unit": "docs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert j["vs_baseline"] is None and j["gpu_launches"] == 0


def test_cuda_arm_has_no_cpu_fallback():
    if torch.cuda.is_available():
        return
    r = run("--workload", "c1", "--steps", "1", "--warmup", "3")
    assert r.returncode != 0 and "no CUDA device" in (r.stderr + r.stdout)
