"""Pins for the oracle's spin-weighted harmonics (oracle O7) -- CPU only.

Each pin is something the paper prints or the mathematics fixes, evaluated by a route that is
NOT the oracle's three-term l-recurrence: the closed forms of App. B, the explicit Wigner-d sum,
textbook Y_lm from scipy, sY_lm derived symbolically with the spin-raising operator (sympy),
the (B.2) inner products and orthonormality (37) by Gauss-Legendre quadrature.
"""
import math
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")
THETAS = [0.05, 0.3, 0.7, 1.1, math.pi / 2, 2.2, 2.9, 3.1]


def _ns():
    return {"sqrt": np.sqrt, "sin": np.sin, "cos": np.cos, "pi": np.pi}


def test_appendix_B_table():
    """PAPER.md:760-762 (B.1): every legible closed form."""
    rows = [l.split(None, 3) for l in open(os.path.join(GOLD, "appB_table.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 27
    for n, l, m, expr in rows:
        n, l, m = int(n), int(l), int(m)
        for t in THETAS:
            want = eval(expr, _ns(), {"t": t})
            got = oracle.spin_P(n, m, 2, t)[l]
            assert abs(got - want) < 2e-15, (n, l, m, t, got, want)


def test_recurrence_equals_explicit_wigner_sum():
    """DESIGN.md reading Q9: P^n_lm = (-1)^n sqrt((2l+1)/4pi) d^l_{m,-n}, explicit sum, l <= 10."""
    for n in range(-3, 4):
        for m in range(-10, 11):
            for t in THETAS:
                got = oracle.spin_P(n, m, 10, t)
                for l in range(0, 11):
                    want = (-1) ** n * math.sqrt((2 * l + 1) / (4 * math.pi)) * oracle.wigner_d_sum(l, m, -n, t)
                    assert abs(got[l] - want) < 1e-13, (n, l, m, t)


def test_scalar_harmonics_match_scipy():
    """n = 0 is the textbook Y_lm (eq. 26): scipy.special.sph_harm_y up to l = 40."""
    from scipy.special import sph_harm_y
    for m in range(-40, 41, 3):
        for t in THETAS:
            got = oracle.spin_P(0, m, 40, t)
            for l in range(abs(m), 41):
                want = sph_harm_y(l, m, t, 0.0).real
                assert abs(got[l] - want) < 5e-13 * max(1.0, abs(want)), (l, m, t)


def test_spin_harmonics_from_spin_raising_operator():
    """sY_lm, l <= 3, all |s| <= l, derived symbolically from the textbook Y_lm with
    eth / eth-bar (Goldberg et al. convention; the paper's n equals that s, App. B)."""
    import sympy as sp
    th, ph = sp.symbols("theta phi", real=True)

    def eth(f, s):
        return -(sp.sin(th) ** s) * (sp.diff(f * sp.sin(th) ** (-s), th) + sp.I / sp.sin(th) * sp.diff(f * sp.sin(th) ** (-s), ph))

    def ethbar(f, s):
        return -(sp.sin(th) ** (-s)) * (sp.diff(f * sp.sin(th) ** s, th) - sp.I / sp.sin(th) * sp.diff(f * sp.sin(th) ** s, ph))

    for l in range(0, 4):
        for m in range(-l, l + 1):
            Y = sp.Ynm(l, m, th, ph).expand(func=True)
            for s in range(-min(l, 3), min(l, 3) + 1):
                f = Y
                if s >= 0:
                    for q in range(s):
                        f = eth(f, q)
                    f = sp.sqrt(sp.factorial(l - s) / sp.factorial(l + s)) * f
                else:
                    for q in range(0, s, -1):
                        f = ethbar(f, q)
                    f = (-1) ** s * sp.sqrt(sp.factorial(l + s) / sp.factorial(l - s)) * f
                fn = sp.lambdify((th, ph), f, "numpy")
                for t in THETAS[1:-1]:
                    want = complex(fn(t, 0.0))
                    got = oracle.spin_P(s, m, 3, t)[l]
                    assert abs(want.imag) < 1e-13
                    assert abs(got - want.real) < 1e-13, (l, m, s, t, got, want)


def test_symmetries_41_47():
    """PAPER.md:356 (eq. 47): P^n_lm = (-1)^{n+m} P^{-n}_{l,-m}; zero below max(|m|,|n|) (eq. 40)."""
    for n in range(-3, 4):
        for m in range(-12, 13):
            for t in THETAS:
                a = oracle.spin_P(n, m, 20, t)
                b = oracle.spin_P(-n, -m, 20, t)
                assert np.max(np.abs(a - (-1) ** (n + m) * b)) < 1e-14
                assert np.all(a[: max(abs(n), abs(m))] == 0)


def _gl(npts=400):
    # Gauss-Legendre in theta itself: the integrands are trigonometric polynomials in theta/2
    # (not polynomials in cos theta when n is odd), for which this converges geometrically.
    x, w = np.polynomial.legendre.leggauss(npts)
    th = np.pi / 2 * (x + 1)
    return th, w * np.pi / 2 * np.sin(th)          # int_0^pi f sin(th) dth = sum w f(th)


def test_inner_products_B2():
    """PAPER.md:768 (B.2); the phi integral gives 2 pi delta_mm'."""
    th, w = _gl()
    for line in open(os.path.join(GOLD, "appB_inner_products.txt")):
        if not line.strip() or line[0] == "#":
            continue
        n1, l1, m1, n2, l2, m2, expr = line.split(None, 6)
        n1, l1, m1, n2, l2, m2 = map(int, (n1, l1, m1, n2, l2, m2))
        want = eval(expr, _ns())
        a = np.array([oracle.spin_P(n1, m1, l1, t)[l1] for t in th])
        b = np.array([oracle.spin_P(n2, m2, l2, t)[l2] for t in th])
        got = 2 * np.pi * np.sum(w * a * b) if m1 == m2 else 0.0
        assert abs(got - want) < 1e-13, (line, got, want)


@pytest.mark.parametrize("n,m", [(0, 0), (0, 5), (1, 0), (1, -3), (-1, 2), (2, 2), (-2, 7), (3, 1), (-3, -4), (3, 30)])
def test_orthonormality_37(n, m):
    """PAPER.md:297 (eq. 37) for fixed n, m: 2 pi int P^n_lm P^n_l'm sin th dth = delta_ll', l <= 95."""
    th, w = _gl(300)
    lmax = 95
    P = np.array([oracle.spin_P(n, m, lmax, t) for t in th])        # [pt, l]
    G = 2 * np.pi * (P * w[:, None]).T @ P
    l0 = max(abs(n), abs(m))
    want = np.diag([1.0 if l >= l0 else 0.0 for l in range(lmax + 1)])
    assert np.max(np.abs(G - want)) < 2e-13


def test_paper_recursion_42_44():
    """PAPER.md:321-336 (eq. 42-44), as printed (reading Q8): Y^n from Y^{n-1} (n>0), Y^{n} from
    Y^{n+1} (n<0).  Checked in the well-conditioned mid-latitudes."""
    def alpha(n, l):
        return math.sqrt((l - n + 1) / (l + n))

    def beta(n, l, m):
        return (1.0 / l) * math.sqrt((2 * l + 1) / (2 * l - 1) * (l + n - 1) * (l * l - m * m) / (l + n))

    for t in [0.6, 1.0, 1.4, 2.0, 2.5]:
        s, c = math.sin(t), math.cos(t)
        for m in range(-6, 7):
            P = {n: oracle.spin_P(n, m, 12, t) for n in range(-3, 4)}
            for l in range(1, 13):
                for n in range(1, 4):
                    if l < max(n, abs(m)):
                        continue
                    up = alpha(n, l) * (m / l - c) / s * P[n - 1][l] + beta(n, l, m) / s * P[n - 1][l - 1]
                    assert abs(up - P[n][l]) < 1e-11, ("42", n, l, m, t)
                    dn = alpha(n, l) * (m / l + c) / s * P[-n + 1][l] - beta(n, l, m) / s * P[-n + 1][l - 1]
                    assert abs(dn - P[-n][l]) < 1e-11, ("43", n, l, m, t)
