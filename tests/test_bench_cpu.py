"""Host-side pieces of bench.py that need no GPU: the paper-style dgemm gradient used as a timing baseline must
compute the same gradient as the oracle (eq. 13-19 against eq. 6-9 naive loops)."""
import numpy as np

import bench
import oracle
import synth


def test_paper_style_gradient_matches_oracle():
    for cid in (1, 2):
        cfg = synth.config(cid)
        u = synth.make_state(cfg)
        _, got = bench.paper_style_cpu_gradient(cfg, u, 1)
        want = oracle.gradient(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"])
        want = np.asarray(want).reshape(got.shape)
        for d in range(3):
            for f in range(u.shape[0]):
                assert np.max(np.abs(got[d, f] - want[d, f])) <= 1e-11 * np.max(np.abs(want[d, f]))


def test_flops_per_unit_totals():
    # gradient 2Nr + 4Ntheta + 2Nphi + 13, filter 5(2L+1)
    for cid, g, f in ((1, 95, 65), (2, 239, 195), (3, 463, 435), (4, 911, 915), (5, 591, 595)):
        fl = bench.flops_per_unit(synth.config(cid))
        assert fl["grad_dphi"] + fl["grad_rtheta"] == g
        assert fl["filt_analysis"] + fl["filt_theta"] + fl["filt_synthesis"] == f


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the oracle arm) on the smallest config: one JSON line with the contract's keys."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=300, check=True).stdout.strip().splitlines()
    assert len(out) == 1
    d = json.loads(out[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["unit"] == bench.UNIT and d["metric"] == bench.METRIC
