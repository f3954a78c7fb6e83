"""Pins of the nested-shell coupling of the oracle (oracle.nested_wave_rhs) -- CPU only.
The paper specifies nothing for nested shells, so the pins are the mathematics of the characteristic coupling:
  * a smooth solution that CROSSES the interface: the coupled RHS equals the analytic time derivative on the interface spheres too
    (to the truncation error), where the single-shell freezing condition is wrong by O(1);
  * one physical outer/inner boundary condition: identical to the single-shell oracle's rows;
  * the evolution of the outgoing pulse through the interface tracks the exact solution as well as a single shell does."""
import numpy as np

import oracle
import synth


def _shells(Nr, Nt, radii):
    return [dict(Nr=Nr, Nt=Nt, Np=2 * Nt, rmin=a, rmax=b) for a, b in zip(radii[:-1], radii[1:])]


def _exact(sh, t, **kw):
    return [synth.wave_exact(dict(s), t, **kw) for s in sh]


def _reverse(us, dudt):
    """time reversal of a solution of the first-order system: (psi, Pi, Phi)(t) -> (psi, -Pi, Phi)(-t): an INGOING pulse"""
    sg_u = np.array([1.0, -1.0, 1.0, 1.0, 1.0])[:, None, None, None]
    return [u * sg_u for u in us], [-d * sg_u for d in dudt]


def test_coupled_rhs_matches_the_analytic_time_derivative_across_the_interface():
    sh = _shells(25, 12, (2.0, 7.0, 12.0))                      # the pulse of W6 sits ON the interface r = 7 at t = 0
    h = 1e-4
    kw = dict(amps=(1.0, 0.8, -0.6))
    us = _exact(sh, 0.0, **kw)
    dudt = [(a - b) / (2 * h) for a, b in zip(_exact(sh, h, **kw), _exact(sh, -h, **kw))]
    n = oracle._unit_normal(12, 24)
    for us_, dudt_, ingoing in ((us, dudt, False), _reverse(us, dudt) + (True,)):
        rhs = oracle.nested_wave_rhs(us_, sh)
        scale = max(np.max(np.abs(d)) for d in dudt_)
        # interior and interface rows of both shells (the physical boundary rows carry the freezing condition: excluded)
        assert np.max(np.abs(rhs[0][..., 1:] - dudt_[0][..., 1:])) < 2e-4 * scale
        assert np.max(np.abs(rhs[1][..., :-1] - dudt_[1][..., :-1])) < 2e-4 * scale
        # both sides agree on the RHS of Pi and of the normal part of Phi on the shared sphere
        assert np.max(np.abs(rhs[0][1, ..., -1] - rhs[1][1, ..., 0])) < 1e-14 * scale
        assert np.max(np.abs(np.sum(n * (rhs[0][2:, ..., -1] - rhs[1][2:, ..., 0]), axis=0))) < 1e-13 * scale
        if ingoing:
            # a single shell's freezing condition on that sphere is NOT the solution: the pulse enters shell 0 through it
            alone = oracle.wave_rhs(us_[0], 25, 12, 24, 2.0, 7.0)
            assert np.max(np.abs(alone[..., -1] - dudt_[0][..., -1])) > 0.2 * scale


def test_characteristic_bookkeeping_of_the_exchange():
    """White noise: on the shared sphere each side keeps the RHS of the characteristic field that leaves it, takes the entering
    one from its neighbour, and keeps its own zero-speed fields; the physical boundaries are those of the single-shell oracle."""
    sh = _shells(9, 6, (1.0, 2.0, 3.5))
    rng = np.random.default_rng(12)
    us = [rng.standard_normal((5, 12, 6, 9)) for _ in sh]
    raw = [oracle.wave_rhs_raw(u, 9, 6, 12, s["rmin"], s["rmax"]) for u, s in zip(us, sh)]
    rhs = oracle.nested_wave_rhs(us, sh)
    n = oracle._unit_normal(6, 12)
    dot = lambda d, k: np.sum(n * d[2:, ..., k], axis=0)
    A, B, a, b = rhs[0], rhs[1], raw[0], raw[1]
    assert np.allclose(A[1, ..., -1] + dot(A, -1), a[1, ..., -1] + dot(a, -1), atol=1e-13)      # U^+ leaves shell 0: own
    assert np.allclose(A[1, ..., -1] - dot(A, -1), b[1, ..., 0] - dot(b, 0), atol=1e-13)        # U^- enters shell 0: neighbour's
    assert np.allclose(B[1, ..., 0] - dot(B, 0), b[1, ..., 0] - dot(b, 0), atol=1e-13)          # U^- leaves shell 1: own
    assert np.allclose(B[1, ..., 0] + dot(B, 0), a[1, ..., -1] + dot(a, -1), atol=1e-13)        # U^+ enters shell 1: neighbour's
    for d, r, k in ((A, a, -1), (B, b, 0)):
        assert np.allclose(d[2:, ..., k] - n * dot(d, k), r[2:, ..., k] - n * dot(r, k), atol=1e-13)   # tangential: own
        assert np.array_equal(d[0, ..., k], r[0, ..., k])                                              # psi: own
    assert np.array_equal(A[..., 1:-1], a[..., 1:-1]) and np.array_equal(B[..., 1:-1], b[..., 1:-1])
    # physical boundaries = the single-shell oracle's rows
    assert np.allclose(A[..., 0], oracle.wave_rhs(us[0], 9, 6, 12, 1.0, 2.0)[..., 0], atol=1e-13)
    assert np.allclose(B[..., -1], oracle.wave_rhs(us[1], 9, 6, 12, 2.0, 3.5)[..., -1], atol=1e-13)


def test_pulse_crosses_the_interface():
    """The outgoing pulse starts on the interface r = 7 and moves into the outer shell (centre at r = 9 at the end); the two-shell
    state agrees with the exact solution to the level a single shell of the same total radial resolution reaches."""
    sh = _shells(17, 10, (2.0, 7.0, 12.0))
    kw = dict(amps=(1.0, 0.8, -0.6))
    c5 = synth.config(5)
    dt = oracle.nested_wave_dt(sh)
    nst = 10
    us = oracle.nested_wave_rk4(_exact(sh, 0.0, **kw), sh, 5, c5["tensors"], dt, nst)
    ex = _exact(sh, nst * dt, **kw)
    scale = max(np.max(np.abs(e)) for e in ex)
    err2 = max(np.max(np.abs(u - e)) for u, e in zip(us, ex))
    one = dict(Nr=33, Nt=10, Np=20, rmin=2.0, rmax=12.0)
    u1 = oracle.wave_rk4(synth.wave_exact(one, 0.0, **kw), 33, 10, 20, 2.0, 12.0, 5, c5["tensors"], dt / 2, 2 * nst)   # its own CFL
    err1 = np.max(np.abs(u1 - synth.wave_exact(one, nst * dt, **kw)))
    assert err2 < 2e-2 * scale and err2 < 5 * err1 + 1e-3 * scale, (err2, err1, scale)
    moved = max(np.max(np.abs(u - e)) for u, e in zip(us, _exact(sh, 0.0, **kw)))
    assert moved > 10 * err2
