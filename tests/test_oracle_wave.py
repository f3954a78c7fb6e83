"""Pins for the oracle's first-order scalar wave system (O13) -- CPU only: the analytic outgoing
multipole solution (closed form), the characteristic structure of the boundary condition, and a
short evolution against the exact solution."""
import numpy as np

import oracle
import synth


def _cfg(Nr, Nt):
    c = synth.config(5)
    c.update(Nr=Nr, Nt=Nt, Np=2 * Nt, L=Nt - 5, npts=Nr * Nt * 2 * Nt)
    return c


def test_exact_solution_satisfies_the_first_order_system():
    """Generator check (closed form): d_t psi = -Pi, and d_t Pi = -div Phi, d_t Phi = -grad Pi hold for
    the analytic fields (time derivative by central differences, space by the oracle gradient)."""
    c = _cfg(33, 24)
    h = 1e-4
    u0 = synth.wave_exact(c, 0.3)
    dudt = (synth.wave_exact(c, 0.3 + h) - synth.wave_exact(c, 0.3 - h)) / (2 * h)
    assert np.max(np.abs(dudt[0] + u0[1])) < 1e-7
    g = oracle.gradient(u0[:1], c["Nr"], c["Nt"], c["Np"], c["rmin"], c["rmax"])[:, 0]
    assert np.max(np.abs(g - u0[2:])) < 2e-3            # Phi_i = d_i psi up to the grid's truncation error


def test_wave_rhs_interior_matches_analytic_time_derivative():
    c = synth.config(5)
    c.update(Nt=32, Np=64)                               # l <= 4 needs little angular resolution
    h = 1e-4
    u0 = synth.wave_exact(c, 0.0)
    dudt = (synth.wave_exact(c, h) - synth.wave_exact(c, -h)) / (2 * h)
    rhs = oracle.wave_rhs(u0, c["Nr"], c["Nt"], c["Np"], c["rmin"], c["rmax"])
    assert np.max(np.abs(rhs - dudt)[..., 1:-1]) < 1e-4 * np.max(np.abs(dudt))   # 2e-5 at config 5


def test_boundary_condition_characteristic_structure():
    """On both boundary shells the incoming field's RHS vanishes, U^- = d_Pi - s.d_Phi = 0, while the
    outgoing U^+ = d_Pi + s.d_Phi, psi and the tangential part of d_Phi keep their interior values."""
    c = _cfg(9, 8)
    rng = np.random.default_rng(2)
    u = rng.standard_normal((5, c["Np"], c["Nt"], c["Nr"]))
    rhs = oracle.wave_rhs(u, c["Nr"], c["Nt"], c["Np"], c["rmin"], c["rmax"])
    g = oracle.gradient(u[1:], c["Nr"], c["Nt"], c["Np"], c["rmin"], c["rmax"])      # [3, 4(Pi,Phi), ...]
    raw = np.stack([-u[1], -(g[0, 1] + g[1, 2] + g[2, 3]), -g[0, 0], -g[1, 0], -g[2, 0]])
    assert np.allclose(rhs[..., 1:-1], raw[..., 1:-1], rtol=0, atol=1e-13)
    th = np.pi * (np.arange(c["Nt"]) + 0.5) / c["Nt"]; ph = 2 * np.pi * np.arange(c["Np"]) / c["Np"]
    PH, TH = np.meshgrid(ph, th, indexing="ij")
    n = np.stack([np.sin(TH) * np.cos(PH), np.sin(TH) * np.sin(PH), np.cos(TH)])
    for k, sg in ((0, -1.0), (c["Nr"] - 1, 1.0)):
        s = sg * n
        d, r = rhs[..., k], raw[..., k]
        sd, sr = np.sum(s * d[2:], axis=0), np.sum(s * r[2:], axis=0)
        assert np.max(np.abs(d[1] - sd)) < 1e-12                                  # incoming frozen
        assert np.max(np.abs((d[1] + sd) - (r[1] + sr))) < 1e-12                  # outgoing kept
        assert np.max(np.abs((d[2:] - s * sd) - (r[2:] - s * sr))) < 1e-12        # tangential kept
        assert np.array_equal(d[0], r[0])


def test_short_evolution_tracks_exact_solution():
    c = _cfg(25, 12)
    Nr, Nt, Np = c["Nr"], c["Nt"], c["Np"]
    dt = oracle.wave_dt(Nr, Nt, Np, c["rmin"], c["rmax"])
    assert abs(oracle.wave_dt(33, 64, 128, 2.0, 12.0) - 0.00964) < 1e-5
    u0 = synth.wave_exact(c, 0.0, amps=(1.0, 0.8, -0.6))
    n = 10
    u = oracle.wave_rk4(u0, Nr, Nt, Np, c["rmin"], c["rmax"], c["L"], c["tensors"], dt, n)
    ex = synth.wave_exact(c, n * dt, amps=(1.0, 0.8, -0.6))
    assert np.max(np.abs(u - ex)) < 2e-2 * np.max(np.abs(ex))
    assert np.max(np.abs(u - u0)) > 10 * np.max(np.abs(u - ex))                       # it actually moved
