"""bench.py on a GPU box: the contract line of the main arm (short run, other legs skipped)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "7", "--warmup", "3", "--no-others",
                          "--no-cpu-baseline", *extra], capture_output=True, text=True, timeout=600, check=True).stdout.strip().splitlines()
    assert len(out) == 1                                   # ONE JSON line on stdout
    return json.loads(out[0])


@pytest.mark.parametrize("extra", [(), ("--no-graph",)])
def test_main_arm_contract_line(extra):
    d = _run(*extra)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in d, key
    assert d["steps"] == 7 and d["warmup"] == 3 and d["n_gpus"] == 1 and d["dtype"] == "f64" and d["scaling"] == "weak"
    assert d["gpu_launches"] > 0 and d["gpu_launches"] % 7 == 0      # kernels per step (counted by the library) x steps
    assert abs(d["value"] - 65 * 96 * 192 * 58 / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    r = d["roofline"]
    assert r["bound"] == "alu" and 0.0 < r["frac"] < 1.0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 58 * 65 * 96 * 192 * 8 and e["d2h_bytes_per_step"] == 4 * e["h2d_bytes_per_step"]
    assert 0.0 < e["value"] < d["value"]                   # host copies inside the timed region can only slow it down
    assert "workload" in d["config"] and "config 4" in d["config"]["workload"]      # the largest single-GPU configuration
    for which in ("gradient", "filter"):                   # each call alone: eager and replayed from a CUDA graph
        c = d["calls"][which]
        assert 0.0 < c["frac_of_fp64_peak"] < 1.0 and c["graph_ms"] is not None and 0.0 < c["graph_frac_of_fp64_peak"] < 1.0
