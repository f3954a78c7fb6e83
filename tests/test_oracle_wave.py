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


# ---- oracle.wave_rk4 is "standard fourth order Runge-Kutta": order and exact one-step amplification ------------
# With an empty tensor list oracle.tensor_filter copies every field through, so wave_rk4 is the bare time integrator of the
# LINEAR system du/dt = A u, A = oracle.wave_rhs (gradient + characteristic boundary condition).
def _rk4_nofilter(u0, c, dt, n):
    return oracle.wave_rk4(u0, c["Nr"], c["Nt"], c["Np"], c["rmin"], c["rmax"], c["L"], [], dt, n)


def test_rk4_one_step_is_the_degree_4_taylor_polynomial_of_the_linear_system():
    """For a linear autonomous system one step of any 4-stage 4th-order Runge-Kutta method is
    u(dt) = (1 + z + z^2/2 + z^3/6 + z^4/24) u(0), z = dt A.  Euler, RK2, or stage weights 1/4,1/4,1/4,1/4 all give a
    different polynomial.  A is applied through oracle.wave_rhs (white-noise data: every mode, both boundaries)."""
    c = _cfg(9, 6)
    Nr, Nt, Np = c["Nr"], c["Nt"], c["Np"]
    u0 = np.random.default_rng(8).standard_normal((5, Np, Nt, Nr))
    dt = 0.7 * oracle.wave_dt(Nr, Nt, Np, c["rmin"], c["rmax"])
    A = lambda v: oracle.wave_rhs(v, Nr, Nt, Np, c["rmin"], c["rmax"])
    term, want = u0.copy(), u0.copy()
    for q in (1, 2, 3, 4):
        term = dt / q * A(term)
        want += term
    got = _rk4_nofilter(u0, c, dt, 1)
    scale = np.max(np.abs(want))
    assert np.max(np.abs(got - want)) < 1e-13 * scale
    # discriminating power: the z^4/24 and z^3/6 terms are far above the tolerance
    assert np.max(np.abs(term)) > 1e-4 * scale
    # two steps compose
    assert np.max(np.abs(_rk4_nofilter(u0, c, dt, 2) - _rk4_nofilter(got, c, dt, 1))) < 1e-13 * scale


def test_rk4_converges_with_fourth_order():
    """Same data to the same final time with dt and dt/2 against a dt/8 reference: the error ratio is 2^4 = 16 (+- 20 %)."""
    c = _cfg(13, 8)
    Nr, Nt, Np = c["Nr"], c["Nt"], c["Np"]
    u0 = synth.wave_exact(c, 0.0, amps=(1.0, 0.8, -0.6))
    dt = 0.5 * oracle.wave_dt(Nr, Nt, Np, c["rmin"], c["rmax"])       # unfiltered, the default lambda = 4 is unstable on this grid
    n = 8
    ref = _rk4_nofilter(u0, c, dt / 8, 8 * n)
    e1 = np.max(np.abs(_rk4_nofilter(u0, c, dt, n) - ref))
    e2 = np.max(np.abs(_rk4_nofilter(u0, c, dt / 2, 2 * n) - ref))
    assert e2 > 1e-11 * np.max(np.abs(ref))              # well above round-off
    assert 0.8 * 16 < e1 / e2 < 1.2 * 16, e1 / e2
