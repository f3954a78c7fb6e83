"""Input data of the single-black-hole test case (eq. A.17): the Schwarzschild metric in Kerr-Schild
form on the grid.  Input generator only -- the given function g_ab(x), no arithmetic of the method (no derivative, no
3+1 split, no Christoffel symbol; those are computed separately by the oracle and by the library)."""
import numpy as np


def grid_xyz(Nr, Nt, Np, rmin, rmax):
    """Cartesian coordinates of the nodes, arrays [Np, Nt, Nr]."""
    k = np.arange(Nr)
    r = 0.5 * (rmax + rmin) - 0.5 * (rmax - rmin) * np.cos(np.pi * k / (Nr - 1))
    th = np.pi * (np.arange(Nt) + 0.5) / Nt
    ph = 2.0 * np.pi * np.arange(Np) / Np
    R, T, P = r[None, None, :], th[None, :, None], ph[:, None, None]
    x = R * np.sin(T) * np.cos(P)
    y = R * np.sin(T) * np.sin(P)
    z = R * np.cos(T) + 0.0 * P
    return x, y, z


def kerr_schild_metric(Nr, Nt, Np, rmin, rmax, M=1.0, center=(0.0, 0.0, 0.0)):
    """g_ab = eta_ab + f l_a l_b, f = 2M/rho, l_a = (1, X_i/rho) (A.17), rho = distance from `center`.
    Returns [10, Np, Nt, Nr] in the order tt,tx,ty,tz,xx,xy,xz,yy,yz,zz."""
    x, y, z = grid_xyz(Nr, Nt, Np, rmin, rmax)
    X = [x - center[0], y - center[1], z - center[2]]
    rho = np.sqrt(X[0] ** 2 + X[1] ** 2 + X[2] ** 2)
    f = 2.0 * M / rho
    l = [np.ones_like(rho)] + [Xi / rho for Xi in X]
    eta = np.diag([-1.0, 1.0, 1.0, 1.0])
    out = []
    for a in range(4):
        for b in range(a, 4):
            out.append(eta[a, b] + f * l[a] * l[b])
    return np.ascontiguousarray(np.stack(out))


def minkowski_metric(Nr, Nt, Np):
    eta = np.diag([-1.0, 1.0, 1.0, 1.0])
    return np.ascontiguousarray(np.stack([np.full((Np, Nt, Nr), eta[a, b]) for a in range(4) for b in range(a, 4)]))


def perturbed_ghg_state(u, amp, seed):
    """u + amp * N(0,1) on every field: a generic (non-stationary, constraint-violating) state for parity tests."""
    rng = np.random.default_rng(seed)
    return u + amp * rng.standard_normal(u.shape)
