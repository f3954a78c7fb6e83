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
    assert _rel(got, want) < TOL * max(1, nsteps)


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
