"""Pins for the oracle's differentiation matrices and Cartesian gradient (O2-O6) -- CPU only.

Pinned to closed forms: exact derivatives of polynomials and trigonometric modes, exact
gradients of polynomials in x, y, z, the paper's example f = r, spectral
convergence.
"""
import numpy as np
import pytest

import oracle


def _xyz(Nr, Nt, Np, rmin, rmax):
    r, th, ph = oracle.grid(Nr, Nt, Np, rmin, rmax)
    R, T, P = np.meshgrid(r, th, ph, indexing="ij")        # [k, i, j]
    to_state = lambda a: np.ascontiguousarray(np.transpose(a, (2, 1, 0)))   # -> [j, i, k]
    x = to_state(R * np.sin(T) * np.cos(P))
    y = to_state(R * np.sin(T) * np.sin(P))
    z = to_state(R * np.cos(T))
    return x, y, z


def test_grid_eq_2_4():
    r, th, ph = oracle.grid(9, 8, 16, 1.0, 3.0)
    assert r[0] == 1.0 and r[-1] == 3.0 and abs(r[4] - 2.0) < 1e-15 and np.all(np.diff(r) > 0)
    assert np.allclose(th, np.pi * (np.arange(8) + 0.5) / 8, rtol=0, atol=1e-15)
    assert np.allclose(ph, 2 * np.pi * np.arange(16) / 16, rtol=0, atol=1e-15)


@pytest.mark.parametrize("N", [9, 17, 33, 65])
def test_cheb_matrix_exact_on_polynomials(N):
    """eq. 9 with the 2/(rmax-rmin) rescaling: d/dr r^p exact for p <= N-1; rows sum to zero."""
    rmin, rmax = 1.8, 10.0
    D = oracle.cheb_diff(N, rmin, rmax)
    r = oracle.grid(N, 2, 4, rmin, rmax)[0]
    s = (r - 0.5 * (rmin + rmax)) / (0.5 * (rmax - rmin))       # in [-1, 1]: keeps powers O(1)
    assert np.max(np.abs(D @ np.ones(N))) < 1e-12 * np.max(np.abs(D))
    for p in range(1, N):
        got = D @ s ** p
        want = p * s ** (p - 1) / (0.5 * (rmax - rmin))
        assert np.max(np.abs(got - want)) < 2e-11 * p * p, p
    # endpoint value of the Chebyshev matrix on [-1,1]: CD_00 = -(2(N-1)^2+1)/6 (known closed form)
    D1 = oracle.cheb_diff(N, -1.0, 1.0)
    assert abs(D1[0, 0] + (2 * (N - 1) ** 2 + 1) / 6.0) < 1e-10
    assert abs(D1[N - 1, N - 1] - (2 * (N - 1) ** 2 + 1) / 6.0) < 1e-10


@pytest.mark.parametrize("n", [16, 48, 96, 192])
def test_fourier_matrix_exact_on_modes(n):
    """eq. 8: exact on sin(qx), cos(qx), q < n/2; the Nyquist mode maps to zero; antisymmetric."""
    D = oracle.fourier_diff(n)
    x = 2 * np.pi * np.arange(n) / n
    assert np.max(np.abs(D + D.T)) == 0.0
    for q in range(0, n // 2):
        assert np.max(np.abs(D @ np.sin(q * x) - q * np.cos(q * x))) < 2e-12 * max(q, 1)
        assert np.max(np.abs(D @ np.cos(q * x) + q * np.sin(q * x))) < 2e-12 * max(q, 1)
    assert np.max(np.abs(D @ np.cos(n // 2 * x))) < 1e-11


def test_theta_derivative_double_cover():
    """d/dtheta of smooth functions on the sphere via the even extension."""
    Nr, Nt, Np = 3, 12, 24
    x, y, z = _xyz(Nr, Nt, Np, 1.0, 2.0)
    r, th, ph = oracle.grid(Nr, Nt, Np, 1.0, 2.0)
    f = (x * z + y)[None]                                   # r^2 sin cos cos(ph) + r sin sin(ph)
    got = oracle.d_theta(f, Nr, Nt, Np)[0]
    R, T, P = [np.transpose(a, (2, 1, 0)) for a in np.meshgrid(r, th, ph, indexing="ij")]
    want = R * R * np.cos(2 * T) * np.cos(P) + R * np.cos(T) * np.sin(P)
    assert np.max(np.abs(got - want)) < 1e-13
    got = oracle.d_phi(f, Nr, Nt, Np)[0]
    want = -R * R * np.sin(T) * np.cos(T) * np.sin(P) + R * np.sin(T) * np.cos(P)
    assert np.max(np.abs(got - want)) < 1e-13


@pytest.mark.parametrize("Nr,Nt", [(9, 8), (17, 24)])
def test_gradient_exact_on_cartesian_polynomials(Nr, Nt):
    """Gradient of polynomials in x, y, z of total degree <= min(Nr-1, Nt-1) is exact (reading Q15)."""
    Np = 2 * Nt
    rmin, rmax = 1.0, 3.0
    x, y, z = _xyz(Nr, Nt, Np, rmin, rmax)
    rng = np.random.default_rng(5)
    deg = min(Nr - 1, Nt - 1, 6)
    f = np.zeros_like(x); fx = np.zeros_like(x); fy = np.zeros_like(x); fz = np.zeros_like(x)
    for a in range(deg + 1):
        for b in range(deg + 1 - a):
            for c in range(deg + 1 - a - b):
                w = rng.standard_normal() / 3.0 ** (a + b + c)
                f += w * x ** a * y ** b * z ** c
                if a: fx += w * a * x ** (a - 1) * y ** b * z ** c
                if b: fy += w * b * x ** a * y ** (b - 1) * z ** c
                if c: fz += w * c * x ** a * y ** b * z ** (c - 1)
    du = oracle.gradient(f[None], Nr, Nt, Np, rmin, rmax)
    scale = max(np.max(np.abs(fx)), np.max(np.abs(fy)), np.max(np.abs(fz)))
    for got, want in zip(du[:, 0], (fx, fy, fz)):
        assert np.max(np.abs(got - want)) < 2e-12 * scale


def test_gradient_of_r_paper_example_and_convergence():
    """f = r gives d_x f = x/r; the error of a smooth non-polynomial
    function falls geometrically with resolution although d(phi)/dx sits half a cell off a pole."""
    errs = []
    for Nr, Nt in [(9, 8), (13, 12), (17, 16), (25, 24)]:
        Np = 2 * Nt
        x, y, z = _xyz(Nr, Nt, Np, 1.0, 3.0)
        r = np.sqrt(x * x + y * y + z * z)
        du = oracle.gradient(r[None], Nr, Nt, Np, 1.0, 3.0)[:, 0]
        assert max(np.max(np.abs(du[0] - x / r)), np.max(np.abs(du[1] - y / r)), np.max(np.abs(du[2] - z / r))) < 1e-12
        f = np.exp(0.4 * x - 0.3 * y + 0.5 * z) / r
        du = oracle.gradient(f[None], Nr, Nt, Np, 1.0, 3.0)[:, 0]
        want = (0.4 - x / r ** 2) * f
        errs.append(np.max(np.abs(du[0] - want)))
    assert errs[0] > 1e-4 and errs[-1] < 1e-10 and all(b < a for a, b in zip(errs, errs[1:]))


def test_gradient_at_matches_full():
    Nr, Nt, Np = 9, 8, 16
    rng = np.random.default_rng(0)
    u = rng.standard_normal((3, Np, Nt, Nr))
    du = oracle.gradient(u, Nr, Nt, Np, 1.0, 3.0)
    samp = np.array([[rng.integers(Nr), rng.integers(Nt), rng.integers(Np), rng.integers(3)] for _ in range(50)], dtype=np.int32)
    got = oracle.gradient_at(u, Nr, Nt, Np, 1.0, 3.0, samp)
    for s, (k, i, j, mu) in enumerate(samp):
        assert np.all(got[s] == du[:, mu, j, i, k])
