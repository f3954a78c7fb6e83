"""Seeded random smooth scalar fields on the shell grid (SURVEY.md 8(d) recipe).

Every stored Cartesian component mu is an independent scalar function
    u^mu[k,i,j] = sum_q sum_{l<=lmax} sum_{|m|<=l} c^mu_{qlm} 2^-l 2^-q T_q(x_k) S_lm(th_i, ph_j),
c ~ N(0,1) from numpy.random.default_rng(seed), drawn per field as an array [q, l, m] (m = -l..l
packed as index m+lmax; entries with |m| > l are drawn and discarded so the stream is layout-
independent).  S_lm = Phat_l^|m|(cos th) cos(m ph) (m >= 0) or sin(|m| ph) (m < 0) with the
ordinary orthonormal associated Legendre functions; T_q Chebyshev polynomials at
x_k = -cos(pi k/(Nr-1)).  Array layout: [field, j, i, k] in C order = p = k + Nr(i + Nt(j + Np mu)).
"""
import numpy as np


def _legendre_hat(lmax, theta):
    """Orthonormal associated Legendre Phat_l^m(cos theta), 0<=m<=l<=lmax: array [l, m, i]."""
    x, s = np.cos(theta), np.sin(theta)
    P = np.zeros((lmax + 1, lmax + 1, theta.size))
    P[0, 0] = np.sqrt(1.0 / (4.0 * np.pi))
    for m in range(1, lmax + 1):
        P[m, m] = -np.sqrt((2.0 * m + 1.0) / (2.0 * m)) * s * P[m - 1, m - 1]
    for m in range(0, lmax):
        P[m + 1, m] = np.sqrt(2.0 * m + 3.0) * x * P[m, m]
    for m in range(0, lmax + 1):
        for l in range(m + 2, lmax + 1):
            a = np.sqrt((4.0 * l * l - 1.0) / (l * l - m * m))
            b = np.sqrt(((l - 1.0) ** 2 - m * m) / (4.0 * (l - 1.0) ** 2 - 1.0))
            P[l, m] = a * (x * P[l - 1, m] - b * P[l - 2, m])
    return P


def scalar_basis(Nr, Nt, Np, lmax):
    theta = np.pi * (np.arange(Nt) + 0.5) / Nt
    phi = 2.0 * np.pi * np.arange(Np) / Np
    xk = -np.cos(np.pi * np.arange(Nr) / (Nr - 1))
    T = np.cos(np.outer(np.arccos(np.clip(xk, -1, 1)), np.arange(Nr)))       # T[k, q]
    return xk, theta, phi, T, _legendre_hat(lmax, theta)


def _synthesise(coef, T, P, phi, decay_l, decay_q):
    """coef [q, l, m+lmax] -> field [j, i, k]."""
    Nr = T.shape[0]
    lmax = P.shape[0] - 1
    Nt = P.shape[2]
    nq = coef.shape[0]
    wl = (2.0 ** (-np.arange(lmax + 1))) if decay_l else np.ones(lmax + 1)
    wq = (2.0 ** (-np.arange(nq, dtype=float))) if decay_q else np.ones(nq)
    c = coef * wq[:, None, None] * wl[None, :, None]
    R = T[:, :nq] @ c.reshape(nq, -1)                                      # [k, (l, m)]
    R = R.reshape(Nr, lmax + 1, 2 * lmax + 1)
    X = np.empty((2 * lmax + 1, Nt, Nr))
    trig = np.empty((phi.size, 2 * lmax + 1))
    for m in range(-lmax, lmax + 1):
        am = abs(m)
        X[m + lmax] = (R[:, am:, m + lmax] @ P[am:, am, :]).T              # [i, k]
        trig[:, m + lmax] = np.cos(am * phi) if m >= 0 else np.sin(am * phi)
    return (trig @ X.reshape(2 * lmax + 1, Nt * Nr)).reshape(phi.size, Nt, Nr)


def make_state(cfg, decay=True, lmax=None, nfields=None, seed=None):
    """The configuration's synthetic state, array [nfields, Np, Nt, Nr] float64."""
    Nr, Nt, Np = cfg["Nr"], cfg["Nt"], cfg["Np"]
    lmax = cfg["lmax"] if lmax is None else lmax
    nf = cfg["nfields"] if nfields is None else nfields
    rng = np.random.default_rng(cfg["seed"] if seed is None else seed)
    _, _, phi, T, P = scalar_basis(Nr, Nt, Np, lmax)
    u = np.empty((nf, Np, Nt, Nr))
    for mu in range(nf):
        coef = rng.standard_normal((Nr, lmax + 1, 2 * lmax + 1))
        for l in range(lmax + 1):                       # discard |m| > l
            coef[:, l, : lmax - l] = 0.0
            coef[:, l, lmax + l + 1:] = 0.0
        u[mu] = _synthesise(coef, T, P, phi, decay, decay)
    return u


def white_state(cfg, nfields=None, seed=0):
    """Test-only: unstructured N(0,1) grid values (every representable mode, no decay)."""
    nf = cfg["nfields"] if nfields is None else nfields
    rng = np.random.default_rng(cfg["seed"] * 7 + seed)
    return rng.standard_normal((nf, cfg["Np"], cfg["Nt"], cfg["Nr"]))
