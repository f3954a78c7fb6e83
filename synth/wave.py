"""Analytic outgoing multipole pulses of the scalar wave equation (config 5 initial data and exact
solution).  Input synthesis only -- none of the method's arithmetic.

    psi = sum_l a_l R_l(t, r) P_l(x,y,z)/r^l,   R_l = sum_{k=0}^{l} (l+k)!/(2^k k! (l-k)!) F^{(l-k)}(t-r) / r^{k+1},
    F(s) = exp(-(s + r_c)^2 / (2 sigma^2))   (pulse centred at r = r_c + t),
P_l harmonic homogeneous polynomials: 1, z, x^2-y^2, xyz, Re (x+iy)^4.   Pi = -d_t psi, Phi_i = d_i psi.
"""
from math import factorial

import numpy as np


def _gauss_derivs(s, rc, sigma, qmax):
    """F^{(q)}(s), q = 0..qmax, by the Hermite recurrence He_{q+1} = z He_q - q He_{q-1}."""
    z = (s + rc) / sigma
    F = np.exp(-0.5 * z * z)
    He = [np.ones_like(z), z]
    for q in range(1, qmax):
        He.append(z * He[q] - q * He[q - 1])
    return [(-1.0 / sigma) ** q * He[q] * F for q in range(qmax + 1)]


def _polys(x, y, z):
    one, zero = np.ones_like(x), np.zeros_like(x)
    P = [one, z, x * x - y * y, x * y * z, x ** 4 - 6 * x * x * y * y + y ** 4]
    dP = [(zero, zero, zero), (zero, zero, one), (2 * x, -2 * y, zero), (y * z, x * z, x * y),
          (4 * x ** 3 - 12 * x * y * y, -12 * x * x * y + 4 * y ** 3, zero)]
    return P, dP


def wave_exact(cfg, t, amps=(1.0, 0.8, -0.6, 0.9, 0.5), rc=7.0, sigma=1.0):
    """u = (psi, Pi, Phi_x, Phi_y, Phi_z) at time t on the grid of cfg: array [5, Np, Nt, Nr]."""
    Nr, Nt, Np = cfg["Nr"], cfg["Nt"], cfg["Np"]
    r = 0.5 * (cfg["rmax"] + cfg["rmin"]) - 0.5 * (cfg["rmax"] - cfg["rmin"]) * np.cos(np.pi * np.arange(Nr) / (Nr - 1))
    th = np.pi * (np.arange(Nt) + 0.5) / Nt
    ph = 2 * np.pi * np.arange(Np) / Np
    PH, TH, R = np.meshgrid(ph, th, r, indexing="ij")
    x, y, z = R * np.sin(TH) * np.cos(PH), R * np.sin(TH) * np.sin(PH), R * np.cos(TH)
    P, dP = _polys(x, y, z)
    lmax = len(amps) - 1
    Fd = _gauss_derivs(t - R, rc, sigma, lmax + 1)
    psi = np.zeros_like(R); Pi = np.zeros_like(R); Phi = [np.zeros_like(R) for _ in range(3)]
    xs = (x, y, z)
    for l, a in enumerate(amps):
        if a == 0.0:
            continue
        Rl = np.zeros_like(R); Rl_t = np.zeros_like(R); Rl_r = np.zeros_like(R)
        for k in range(l + 1):
            c = factorial(l + k) / (2 ** k * factorial(k) * factorial(l - k))
            Rl += c * Fd[l - k] / R ** (k + 1)
            Rl_t += c * Fd[l - k + 1] / R ** (k + 1)
            Rl_r += c * (-Fd[l - k + 1] / R ** (k + 1) - (k + 1) * Fd[l - k] / R ** (k + 2))
        ang = P[l] / R ** l
        psi += a * Rl * ang
        Pi += -a * Rl_t * ang
        for c in range(3):
            dang = dP[l][c] / R ** l - l * P[l] * xs[c] / R ** (l + 2)
            Phi[c] += a * (Rl_r * xs[c] / R * ang + Rl * dang)
    return np.stack([psi, Pi, Phi[0], Phi[1], Phi[2]])
