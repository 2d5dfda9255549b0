"""-m "not gpu": bench.py's reference arm (the CPU oracle) runs here and prints the contract's JSON line;
the product arm refuses to run without a CUDA device instead of falling back to the CPU."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(args, timeout=600):
    env = dict(os.environ, OMP_NUM_THREADS="4")
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                          timeout=timeout, env=env, cwd=ROOT)


def test_reference_arm_prints_contract_line():
    p = run(["--impl", "reference", "--config", "1", "--steps", "2", "--warmup", "1", "--precision", "f64"])
    assert p.returncode == 0, p.stderr[-2000:]
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "pcg_iterations_per_s" and line["unit"] == "iterations/s"
    assert line["higher_is_better"] is True and line["data"] == "synthetic" and line["steps"] == 2 and line["warmup"] == 1
    assert line["value"] > 0 and line["config"]["workload"].startswith("config1_33^3_f64")
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == {"value": line["value"], "unit": "iterations/s", "h2d_bytes_per_step": 0,
                           "d2h_bytes_per_step": 0}
    assert line["vs_baseline"] is None


def test_product_arm_has_no_cpu_fallback():
    import torch

    if torch.cuda.is_available():
        import pytest

        pytest.skip("a CUDA device is present")
    p = run(["--config", "1", "--steps", "1", "--warmup", "1"])
    assert p.returncode != 0
    assert "no CPU fallback" in (p.stderr + p.stdout)
