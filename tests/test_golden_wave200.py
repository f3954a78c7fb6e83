"""The stored oracle run of config 5's 200 RK4 steps (tests/golden/wave200_*.npz, written by tests/golden/make_wave200.py from
oracle/ and synth/ only) must belong to the oracle as it stands, and must be a solution: it tracks the exact outgoing-multipole
solution at truncation level.  CPU only; the GPU comparison is tests/test_gpu_wave.py."""
import importlib.util
import os

import numpy as np
import pytest

import synth

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _mk():
    spec = importlib.util.spec_from_file_location("make_wave200", os.path.join(HERE, "make_wave200.py"))
    mk = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mk)
    return mk


@pytest.mark.parametrize("variant", ["clean", "noise"])
def test_stored_oracle_run_is_current_and_tracks_the_exact_solution(variant):
    mk = _mk()
    gold = np.load(os.path.join(HERE, f"wave200_{variant}.npz"))
    assert str(gold["key"]) == mk.golden_key(variant), "stale: rerun tests/golden/make_wave200.py " + variant
    c = synth.config(5)
    idx, dt = gold["idx"], float(gold["dt"])
    assert idx.shape == (5 * c["Nr"] * mk.NSAMP_PER_RADIUS, 4)
    assert len({(f, k) for f, _, _, k in idx.tolist()}) == 5 * c["Nr"]          # every radius of every field is sampled
    for cp in mk.CHECKPOINTS:
        ex = synth.wave_exact(c, cp * dt)
        val = ex[idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3]]
        scale = np.max(np.abs(ex))
        assert np.max(np.abs(gold[f"val_{cp}"] - val)) < 1e-2 * scale           # truncation-level agreement (boundary condition acting on the tails)
        assert np.all(np.abs(gold[f"maxabs_{cp}"] - np.max(np.abs(ex.reshape(5, -1)), axis=1)) < 2e-2 * scale)
