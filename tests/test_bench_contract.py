"""The JSON line `bench.py` prints: keys the driver reads, for the reference arm (the oracle on the host cores; runs without a
GPU) and for the library's own arm (one B200).  Small sizes: this checks the contract, not the numbers."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
             "dtype", "data", "config", "e2e", "gpu_launches", "cpu_baseline"}


def _run(args, timeout):
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True, timeout=timeout, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, res.stdout[-2000:]                       # exactly ONE JSON line
    return json.loads(lines[0])


def test_reference_arm_line_runs_the_oracle_on_the_host_and_names_the_same_config():
    d = _run(["--impl", "reference", "--n", "256", "--steps", "2", "--warmup", "1"], 300)
    assert d["impl"] == "reference" and BASE_KEYS <= set(d)
    assert d["steps"] == 2 and d["warmup"] == 1 and d["n_gpus"] == 1 and d["higher_is_better"] is True
    assert d["unit"] == "TFLOP/s" and d["value"] > 0 and d["vs_baseline"] is None and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    # the same `config` object as the library's arm prints for the same arguments (the driver compares them)
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    ns = argparse.Namespace(workload="config4", n=256, mode="split16", option=[], stop="paper", max_iter=20)
    assert d["config"] == bench.bench_config(ns, 1)
    assert d["config"]["workload"] == "config4_n256"


@pytest.mark.gpu
def test_library_arm_line_quick_mode():
    d = _run(["--n", "1024", "--steps", "3", "--warmup", "3", "--quick"], 600)
    assert BASE_KEYS | {"roofline", "clocks", "iters", "err_history", "flags"} <= set(d) and "impl" not in d
    assert d["steps"] == 3 and d["warmup"] == 3 and d["n_gpus"] == 1 and d["value"] > 0 and d["gpu_launches"] > 0
    assert d["config"]["workload"] == "config4_n1024" and d["config"]["mode"] == "split16" and d["data"] == "synthetic"
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 2 * 1024 * 1024 * 4 and e["d2h_bytes_per_step"] >= 1024 * 1024 * 4
    r = d["roofline"]
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and r["peak"] > 0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
