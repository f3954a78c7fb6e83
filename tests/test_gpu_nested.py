"""GPU parity of the nested-shell path: sp_rhs_wave_shell + sp_wave_interface and the
RK4 driver against oracle.nested_wave_rhs / nested_wave_rk4 (1e-12 relative, max-norm per field), and the pulse crossing the
interface against the exact solution."""
import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu
TOL = 1e-12


def _rel(a, b):
    a = a.reshape(a.shape[0], -1); b = b.reshape(a.shape)
    return float(np.max(np.max(np.abs(a - b), axis=1) / np.max(np.abs(b), axis=1)))


def _setup(Nrs, Nt, radii, L):
    from paper_1104_3408_b200 import Shell
    sh = [dict(Nr=Nr, Nt=Nt, Np=2 * Nt, rmin=a, rmax=b) for Nr, a, b in zip(Nrs, radii[:-1], radii[1:])]
    gs = [Shell(s["Nr"], s["Nt"], s["Np"], s["rmin"], s["rmax"], L) for s in sh]
    return sh, gs


def test_nested_rhs_parity_three_shells_of_different_radial_resolution():
    import torch
    from paper_1104_3408_b200.nested import NestedWaveRK4
    sh, gs = _setup((9, 17, 12), 12, (1.5, 3.0, 6.0, 8.5), 7)
    rng = np.random.default_rng(31)
    us = [rng.standard_normal((5, s["Np"], s["Nt"], s["Nr"])) for s in sh]          # white noise: every mode, every boundary row
    rk = NestedWaveRK4(gs, synth.config(5)["tensors"])
    got = rk.rhs([torch.from_numpy(u).cuda() for u in us])
    want = oracle.nested_wave_rhs(us, sh)
    for g, w in zip(got, want):
        assert _rel(g.cpu().numpy(), w) < TOL
    assert abs(rk.dt() - oracle.nested_wave_dt(sh)) < 1e-15


def test_interface_argument_checks():
    import torch
    from paper_1104_3408_b200 import Shell
    from paper_1104_3408_b200.binding import SpError
    a, b, c = Shell(9, 8, 16, 1.0, 2.0, 3), Shell(9, 8, 16, 2.0, 3.0, 3), Shell(9, 6, 12, 2.0, 3.0, 1)
    da = torch.zeros((5, 16, 8, 9), dtype=torch.float64, device="cuda")
    db = torch.zeros_like(da)
    Shell.wave_interface(a, da, b, db)
    with pytest.raises(SpError):
        Shell.wave_interface(b, db, a, da)                       # radii do not match in this order
    with pytest.raises(SpError):
        Shell.wave_interface(a, da, c, torch.zeros((5, 12, 6, 9), dtype=torch.float64, device="cuda"))   # different angular grid
    with pytest.raises(SpError):
        Shell.wave_interface(a, da, a, da)


@pytest.mark.parametrize("graph", [False, True])
def test_nested_rk4_parity_with_oracle(graph):
    """Two shells, 6 RK4 steps with the Yn filter per shell and substep, pulse on the interface + 1e-6 white noise."""
    import torch
    from paper_1104_3408_b200.nested import NestedWaveRK4
    sh, gs = _setup((17, 13), 12, (2.0, 7.0, 12.0), 7)
    c5 = synth.config(5)
    rng = np.random.default_rng(32)
    us = [synth.wave_exact(s, 0.0) + 1e-6 * rng.standard_normal((5, s["Np"], s["Nt"], s["Nr"])) for s in sh]
    rk = NestedWaveRK4(gs, c5["tensors"])
    dt = rk.dt()
    got = rk.evolve([torch.from_numpy(u).cuda() for u in us], dt, 6, graph=graph)
    want = oracle.nested_wave_rk4(us, sh, 7, c5["tensors"], dt, 6)
    for g, w in zip(got, want):
        assert _rel(g.cpu().numpy(), w) < TOL


def test_pulse_crosses_the_interface_on_the_gpu():
    """Config-5 angular grid, two shells of 33 radial points: the outgoing pulse starts on the interface r = 7; at t ~ 2 the state
    agrees with the exact solution at truncation level (as the single shell of config 5 does)."""
    import torch
    from paper_1104_3408_b200.nested import NestedWaveRK4
    sh, gs = _setup((33, 33), 32, (2.0, 7.0, 12.0), 27)
    rk = NestedWaveRK4(gs, synth.config(5)["tensors"])
    dt = rk.dt()
    n = int(2.0 / dt)
    us = rk.evolve([torch.from_numpy(synth.wave_exact(s, 0.0)).cuda() for s in sh], dt, n, graph=True)
    ex = [synth.wave_exact(s, n * dt) for s in sh]
    scale = max(np.max(np.abs(e)) for e in ex)
    for u, e in zip(us, ex):
        assert np.max(np.abs(u.cpu().numpy() - e)) < 1e-2 * scale
