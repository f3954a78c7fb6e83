"""GPU parity for the first-order scalar wave system (config 5): RHS and RK4 loop against the oracle
(1e-12 relative, max-norm per field) and the full 200-step run against the exact solution."""
import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu
TOL = 1e-12


def _rel(a, b):
    a = a.reshape(a.shape[0], -1); b = b.reshape(a.shape)
    return float(np.max(np.max(np.abs(a - b), axis=1) / np.max(np.abs(b), axis=1)))


def _shell(c):
    from paper_1104_3408_b200 import Shell
    return Shell(c["Nr"], c["Nt"], c["Np"], c["rmin"], c["rmax"], c["L"])


def test_wave_rhs_parity_config5():
    import torch
    c = synth.config(5)
    u = synth.wave_exact(c, 0.0)
    got = _shell(c).rhs_first_order_wave(torch.from_numpy(u).cuda()).cpu().numpy()
    want = oracle.wave_rhs(u, c["Nr"], c["Nt"], c["Np"], c["rmin"], c["rmax"])
    assert _rel(got, want) < TOL
    rng = np.random.default_rng(1)
    u = rng.standard_normal(u.shape)                      # white noise: every mode, both boundaries
    got = _shell(c).rhs_first_order_wave(torch.from_numpy(u).cuda()).cpu().numpy()
    want = oracle.wave_rhs(u, c["Nr"], c["Nt"], c["Np"], c["rmin"], c["rmax"])
    assert _rel(got, want) < TOL


@pytest.mark.parametrize("shape,nsteps,noise", [((17, 12, 24), 25, 1e-6), ((33, 64, 128), 2, 1e-6)])
def test_rk4_parity_with_oracle(shape, nsteps, noise):
    """RK4 + 4 filters per step; 1e-6 white noise on top of the pulse so that the filter's truncation
    acts inside the loop (the clean data never leaves l <= 4)."""
    import torch
    from paper_1104_3408_b200.wave import WaveRK4, wave_dt
    c = synth.config(5)
    c.update(Nr=shape[0], Nt=shape[1], Np=shape[2], L=shape[1] - 5)
    Nr, Nt, Np = shape
    u0 = synth.wave_exact(c, 0.0) + noise * np.random.default_rng(3).standard_normal((5, Np, Nt, Nr))
    dt = wave_dt(Nr, Nt, Np, c["rmin"], c["rmax"])
    assert abs(dt - oracle.wave_dt(Nr, Nt, Np, c["rmin"], c["rmax"])) < 1e-15
    got = WaveRK4(_shell(c), c["tensors"]).evolve(torch.from_numpy(u0).cuda(), dt, nsteps).cpu().numpy()
    want = oracle.wave_rk4(u0, Nr, Nt, Np, c["rmin"], c["rmax"], c["L"], c["tensors"], dt, nsteps)
    assert _rel(got, want) < TOL          # flat: SURVEY.md W7 measured a round-off sensitivity of 6e-15 after 200 steps


def test_config5_200_steps_against_exact_solution():
    import torch
    from paper_1104_3408_b200.wave import WaveRK4, wave_dt
    c = synth.config(5)
    Nr, Nt, Np = c["Nr"], c["Nt"], c["Np"]
    dt = wave_dt(Nr, Nt, Np, c["rmin"], c["rmax"])
    u = torch.from_numpy(synth.wave_exact(c, 0.0)).cuda()
    out = WaveRK4(_shell(c), c["tensors"]).evolve(u, dt, 200).cpu().numpy()
    ex = synth.wave_exact(c, 200 * dt)
    assert np.all(np.isfinite(out))
    assert np.max(np.abs(out - ex)) < 1e-2 * np.max(np.abs(ex))      # truncation-level check


@pytest.mark.parametrize("variant", ["clean", "noise"])
def test_config5_200_steps_against_the_stored_oracle_run(variant):
    """Config 5's own workload (BASELINE.json: 33 x 64 x 128, 200 RK4 steps, BC + Yn filter each substep) against the ORACLE's
    run of the same 200 steps, 1e-12 relative to each field's max-norm, after 100 and after 200 steps.  The oracle run
    (~20 min on 8 cores) is stored by tests/golden/make_wave200.py (imports oracle/ and synth/ only): a stratified sample of
    9 900 values (every radius of every field) plus per-field max-norms; `key` ties the file to the oracle sources.
    "noise" adds 1e-6 white noise so that the filter truncates inside the loop (the clean data never leaves l <= 4)."""
    import importlib.util
    import os
    import torch
    from paper_1104_3408_b200.wave import WaveRK4, wave_dt
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_wave200", os.path.join(here, "make_wave200.py"))
    mk = importlib.util.module_from_spec(spec); spec.loader.exec_module(mk)
    gold = np.load(os.path.join(here, f"wave200_{variant}.npz"))
    assert str(gold["key"]) == mk.golden_key(variant), "stored oracle run is stale: rerun tests/golden/make_wave200.py"
    c, u0 = mk.initial_data(variant)
    Nr, Nt, Np = c["Nr"], c["Nt"], c["Np"]
    dt = wave_dt(Nr, Nt, Np, c["rmin"], c["rmax"])
    assert abs(dt - float(gold["dt"])) < 1e-16
    idx = gold["idx"]
    rk = WaveRK4(_shell(c), c["tensors"])
    u = torch.from_numpy(u0).cuda()
    done = 0
    for cp in mk.CHECKPOINTS:
        u = rk.evolve(u, dt, cp - done) if done == 0 else _continue(rk, u, dt, cp - done)
        done = cp
        got = u.cpu().numpy()
        fmax = gold[f"maxabs_{cp}"]
        assert np.max(np.abs(np.max(np.abs(got.reshape(5, -1)), axis=1) - fmax) / fmax) < TOL
        val = got[idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3]]
        err = np.abs(val - gold[f"val_{cp}"]) / fmax[idx[:, 0]]
        assert err.max() < TOL, (variant, cp, err.max(), idx[np.argmax(err)])


def _continue(rk, u, dt, n):
    """n more RK4 steps WITHOUT evolve()'s initial filter (the stored oracle run is one uninterrupted loop)."""
    for _ in range(n):
        rk._step(u, dt)
    return u


def test_rk4_stage_kernel_and_aliasing_rules():
    """sp_rk4_stage (row W3): acc_out = acc_in + c_acc k, stage_out = u + c_stage k, each rounded once per operation
    (an FMA contraction of c*k + a is within 1 ulp of the two-step value)."""
    import torch
    from paper_1104_3408_b200 import Shell
    from paper_1104_3408_b200.binding import SpError
    rng = np.random.default_rng(5)
    n = 100003                                                            # ragged tail
    u, k, acc = (rng.standard_normal(n) for _ in range(3))
    du, dk, dacc = (torch.from_numpy(x).cuda() for x in (u, k, acc))
    dst = torch.zeros(n, dtype=torch.float64, device="cuda")
    dout = torch.zeros_like(dst)
    Shell.rk4_stage(du, dk, dacc, dout, dst, 0.125, 0.5)
    assert np.max(np.abs(dout.cpu().numpy() - (acc + 0.125 * k))) <= 4e-16 * np.max(np.abs(acc))
    assert np.max(np.abs(dst.cpu().numpy() - (u + 0.5 * k))) <= 4e-16 * np.max(np.abs(u))
    Shell.rk4_stage(du, dk, du, dacc, dst, 0.25, 1.0)                     # first stage: acc_in = u
    assert np.max(np.abs(dacc.cpu().numpy() - (u + 0.25 * k))) <= 4e-16 * np.max(np.abs(u))
    want = dacc.cpu().numpy() + 0.3 * k
    Shell.rk4_stage(du, dk, dacc, du, None, 0.3, 0.0)                     # last stage: new state over u, no stage array
    assert np.max(np.abs(du.cpu().numpy() - want)) <= 4e-16 * np.max(np.abs(want))
    for bad in ((du, dk, dacc, dacc, du), (du, dk, dacc, dk, dst), (du, dk, dacc, dst, dst)):
        with pytest.raises(SpError):
            Shell.rk4_stage(*bad, 0.1, 0.1)


def test_rk4_graph_replay_is_bit_identical_to_eager():
    import torch
    from paper_1104_3408_b200.wave import WaveRK4, wave_dt
    c = synth.config(5)
    c.update(Nr=17, Nt=12, Np=24, L=7)
    u0 = synth.wave_exact(c, 0.0) + 1e-6 * np.random.default_rng(4).standard_normal((5, 24, 12, 17))
    dt = wave_dt(17, 12, 24, c["rmin"], c["rmax"])
    sh = _shell(c)
    a = WaveRK4(sh, c["tensors"]).evolve(torch.from_numpy(u0).cuda(), dt, 7).cpu().numpy()
    rk = WaveRK4(sh, c["tensors"])
    ub = torch.from_numpy(u0).cuda()
    b = rk.evolve(ub, dt, 3, graph=True)
    b = rk.evolve(ub, dt, 4, graph=True).cpu().numpy()                    # second call reuses the captured step
    # evolve() filters its input first; the filter is idempotent only to round-off, so compare to round-off, not bits
    assert _rel(b, a) < 1e-13
    ub2 = torch.from_numpy(u0).cuda()
    b2 = WaveRK4(sh, c["tensors"]).evolve(ub2, dt, 7, graph=True).cpu().numpy()
    assert np.array_equal(b2, a)
