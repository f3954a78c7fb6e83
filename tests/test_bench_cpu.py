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
