"""ctypes binding of the CPU oracle (oracle/sp_oracle.c).

TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package; the product (paper_1104_3408_b200) never does.
The oracle is plain C with long-double accumulation written from PAPER.md; see the header of
sp_oracle.c for what each function follows and how it is pinned.
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

_lib = None
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_wigner_d_sum.restype = C.c_double
        _lib.orc_wigner_d_sum.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double]
        _lib.orc_synthesis_matrix.restype = C.c_int
        _lib.orc_ncomp.restype = C.c_int
    return _lib


def set_threads(n: int) -> None:
    """Number of OpenMP threads the oracle may use (its loops over fields/spheres)."""
    os.environ["OMP_NUM_THREADS"] = str(n)
    try:
        omp = C.CDLL("libgomp.so.1")
        omp.omp_set_num_threads(int(n))
    except OSError:
        pass


def grid(Nr, Nt, Np, rmin, rmax):
    r, th, ph = np.zeros(Nr), np.zeros(Nt), np.zeros(Np)
    lib().orc_grid(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_double(rmin), C.c_double(rmax),
                   r.ctypes, th.ctypes, ph.ctypes)
    return r, th, ph


def cheb_diff(N, rmin, rmax):
    D = np.zeros((N, N))
    lib().orc_cheb_diff(C.c_int(N), C.c_double(rmin), C.c_double(rmax), D.ctypes)
    return D


def fourier_diff(n):
    D = np.zeros((n, n))
    lib().orc_fourier_diff(C.c_int(n), D.ctypes)
    return D


def _state(u, Nr, Nt, Np):
    u = np.ascontiguousarray(u, dtype=np.float64)
    nf = u.size // (Nr * Nt * Np)
    assert nf * Nr * Nt * Np == u.size
    return u, nf


def d_r(u, Nr, Nt, Np, rmin, rmax):
    u, nf = _state(u, Nr, Nt, Np)
    out = np.empty_like(u)
    lib().orc_dr(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_int(nf), C.c_double(rmin), C.c_double(rmax),
                 u.ctypes, out.ctypes)
    return out


def d_theta(u, Nr, Nt, Np):
    u, nf = _state(u, Nr, Nt, Np)
    out = np.empty_like(u)
    lib().orc_dtheta(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_int(nf), u.ctypes, out.ctypes)
    return out


def d_phi(u, Nr, Nt, Np):
    u, nf = _state(u, Nr, Nt, Np)
    out = np.empty_like(u)
    lib().orc_dphi(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_int(nf), u.ctypes, out.ctypes)
    return out


def gradient(u, Nr, Nt, Np, rmin, rmax):
    """u: [nf, Np, Nt, Nr] (C order; r fastest) -> du: [3, nf, Np, Nt, Nr] = d/dx, d/dy, d/dz."""
    u, nf = _state(u, Nr, Nt, Np)
    du = np.empty((3, nf, Np, Nt, Nr))
    lib().orc_gradient(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_int(nf), C.c_double(rmin), C.c_double(rmax),
                       u.ctypes, du.ctypes)
    return du


def gradient_at(u, Nr, Nt, Np, rmin, rmax, samples):
    """samples: int array [ns, 4] of (k, i, j, mu) -> [ns, 3] gradient values."""
    u, nf = _state(u, Nr, Nt, Np)
    s = np.ascontiguousarray(samples, dtype=np.int32)
    out = np.empty((s.shape[0], 3))
    lib().orc_gradient_at(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_int(nf), C.c_double(rmin), C.c_double(rmax),
                          u.ctypes, C.c_int(s.shape[0]), s.ctypes, out.ctypes)
    return out


def wigner_d_sum(l, mp, m, th):
    return lib().orc_wigner_d_sum(l, mp, m, float(th))


def spin_P(n, m, lmax, th):
    """P^n_{lm}(th) for l = 0..lmax (eq. 46)."""
    out = np.zeros(lmax + 1)
    lib().orc_spin_P(C.c_int(n), C.c_int(m), C.c_int(lmax), C.c_double(th), out.ctypes)
    return out


def synthesis_matrix(N, n, m):
    l0 = max(abs(n), abs(m))
    if N - l0 <= 0:
        return np.zeros((N, 0))
    P = np.zeros((N, N - l0))
    lib().orc_synthesis_matrix(C.c_int(N), C.c_int(n), C.c_int(m), P.ctypes)
    return P


def filter_matrix(N, L, n, m):
    F = np.zeros((N, N))
    lib().orc_filter_matrix(C.c_int(N), C.c_int(L), C.c_int(n), C.c_int(m), F.ctypes)
    return F


def spin_analysis(N, n, m, s):
    l0 = max(abs(n), abs(m))
    s = np.ascontiguousarray(s, dtype=np.float64)
    c = np.zeros(max(N - l0, 0))
    lib().orc_spin_analysis(C.c_int(N), C.c_int(n), C.c_int(m), s.ctypes, c.ctypes)
    return c


def spin_filter_sphere(N, L, n, g):
    """g: complex [J=2N, N] (index [j, i]) -> filtered complex array of the same shape."""
    g = np.asarray(g)
    gre = np.ascontiguousarray(g.real, dtype=np.float64)
    gim = np.ascontiguousarray(g.imag if np.iscomplexobj(g) else np.zeros_like(gre), dtype=np.float64)
    ore, oim = np.empty_like(gre), np.empty_like(gre)
    lib().orc_spin_filter_sphere(C.c_int(N), C.c_int(L), C.c_int(n), gre.ctypes, gim.ctypes, ore.ctypes, oim.ctypes)
    return ore + 1j * oim


def ncomp(rank, dims, sym):
    d = np.ascontiguousarray(list(dims) + [0] * (3 - len(dims)), dtype=np.int32)
    return lib().orc_ncomp(C.c_int(rank), d.ctypes, C.c_int(sym[0]), C.c_int(sym[1]))


def tensor_filter(u, Nr, Nt, Np, L, tensors, ksel=-1):
    """Yn tensor filter.  tensors: list of dicts {rank, dims (len rank, 3|4), sym (a,b)|(-1,-1),
    fields [stored components in canonical order]}.  Returns the filtered state (same shape);
    fields in no tensor are copied through.  ksel >= 0: only that radius is filtered."""
    u, nf = _state(u, Nr, Nt, Np)
    out = np.empty_like(u)
    nt = len(tensors)
    rank = np.array([t["rank"] for t in tensors], dtype=np.int32)
    dims = np.zeros((nt, 3), dtype=np.int32)
    sym = np.full((nt, 2), -1, dtype=np.int32)
    foff = np.zeros(nt + 1, dtype=np.int32)
    fl = []
    for q, t in enumerate(tensors):
        for a, d in enumerate(t["dims"]):
            dims[q, a] = d
        sym[q] = t.get("sym", (-1, -1))
        assert len(t["fields"]) == ncomp(t["rank"], t["dims"], sym[q]), "component count mismatch"
        fl += list(t["fields"])
        foff[q + 1] = len(fl)
    fields = np.array(fl if fl else [0], dtype=np.int32)
    lib().orc_tensor_filter(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_int(L), C.c_int(nf), u.ctypes, out.ctypes,
                            C.c_int(nt), rank.ctypes, dims.ctypes, sym.ctypes, foff.ctypes, fields.ctypes,
                            C.c_int(ksel))
    return out


def wave_rhs(u, Nr, Nt, Np, rmin, rmax):
    """RHS of the first-order scalar wave system with the freezing boundary condition (O13)."""
    u, nf = _state(u, Nr, Nt, Np)
    assert nf == 5
    out = np.empty_like(u)
    lib().orc_wave_rhs(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_double(rmin), C.c_double(rmax), u.ctypes, out.ctypes)
    return out


def wave_dt(Nr, Nt, Np, rmin, rmax, lam=4.0):
    """dt = lambda * min(dx) (eq. 63; reading W4): min over the radial spacing at the
    inner boundary and the azimuthal spacing on the innermost shell next to the pole."""
    r, th, ph = grid(Nr, Nt, Np, rmin, rmax)
    dphi = 2.0 * r[0] * np.sin(th[0]) * np.sin(np.pi / Np)
    return lam * min(r[1] - r[0], dphi)


def wave_rk4(u, Nr, Nt, Np, rmin, rmax, L, tensors, dt, nsteps, on_step=None):
    """Classical RK4 with the Yn filter applied to the initial data, to every stage
    state before its RHS and to the final combination: 4 filters per step (reading W5).
    on_step(step, u), if given, is called after every completed step (observation only: snapshots of a long run)."""
    F = lambda v: tensor_filter(v, Nr, Nt, Np, L, tensors)
    R = lambda v: wave_rhs(v, Nr, Nt, Np, rmin, rmax)
    u = F(np.array(u, dtype=np.float64))
    for step in range(1, nsteps + 1):
        k1 = R(u)
        k2 = R(F(u + 0.5 * dt * k1))
        k3 = R(F(u + 0.5 * dt * k2))
        k4 = R(F(u + dt * k3))
        u = F(u + dt / 6.0 * (k1 + 2.0 * k2 + 2.0 * k3 + k4))
        if on_step is not None:
            on_step(step, u)
    return u


# ---- GHG right-hand side (oracle/ghg_oracle.c; Appendix A) ----
def ghg_rhs(u, du, H, dH, Nr, Nt, Np, rmin, rmax, bc_outer=False):
    """(A.8)-(A.10) for the 50-field state u with its Cartesian gradient du [3,50], gauge source H [4] and dH [3,4];
    bc_outer: freezing condition (A.20)-(A.21) on the shell k = Nr-1."""
    u, nf = _state(u, Nr, Nt, Np)
    assert nf == 50
    du = np.ascontiguousarray(du, dtype=np.float64).reshape(3, 50, Np, Nt, Nr)
    H = np.ascontiguousarray(H, dtype=np.float64).reshape(4, Np, Nt, Nr)
    dH = np.ascontiguousarray(dH, dtype=np.float64).reshape(3, 4, Np, Nt, Nr)
    out = np.empty_like(u)
    bad = lib().orc_ghg_rhs(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), C.c_double(rmin), C.c_double(rmax), u.ctypes, du.ctypes,
                            H.ctypes, dH.ctypes, C.c_int(1 if bc_outer else 0), out.ctypes)
    if bad:
        raise ValueError(f"metric not Lorentzian/invertible at {bad} points")
    return out


def ghg_init(g, Nr, Nt, Np, rmin, rmax):
    """Initial data of PAPER.md:732-737 from a metric g_ab [10] with d_t g_ab = 0: d_iab = numerical gradient of g_ab,
    k_ab by (A.6), H_a = -Gamma_a (A.18), dH = numerical gradient of H.  Returns u [50], H [4], dH [3,4]."""
    g, nf = _state(g, Nr, Nt, Np)
    assert nf == 10
    u = np.zeros((50, Np, Nt, Nr))
    u[:10] = g
    u[20:] = gradient(g, Nr, Nt, Np, rmin, rmax).reshape(30, Np, Nt, Nr)
    H = np.zeros((4, Np, Nt, Nr))
    bad = lib().orc_ghg_init(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), u.ctypes, H.ctypes)
    if bad:
        raise ValueError(f"metric not Lorentzian/invertible at {bad} points")
    dH = gradient(H, Nr, Nt, Np, rmin, rmax).reshape(3, 4, Np, Nt, Nr)
    return u, H, dH


def ghg_lapse_shift(u, Nr, Nt, Np):
    """alpha, beta^i, gamma^{ij} (xx,xy,xz,yy,yz,zz) of (A.4)-(A.5): [10] state-shaped."""
    u, nf = _state(u, Nr, Nt, Np)
    out = np.zeros((10, Np, Nt, Nr))
    lib().orc_ghg_lapse_shift(C.c_int(Nr), C.c_int(Nt), C.c_int(Np), u.ctypes, out.ctypes)
    return out


# ---- nested shells (DESIGN.md section 11 readings N1-N4) ----
# The paper names domain decomposition into nested shells as future work and specifies nothing.  Reading: shells
# [R_a, R_a+1] share their interface spheres and the angular grid (the interface points coincide, no interpolation); each shell
# is evolved as in the single-shell case and the shells are coupled through the characteristic fields of (A.13)-(A.16)
# on the shared sphere: with n = r^, U^+ = Pi + n.Phi moves outward and U^- = Pi - n.Phi inward; each side
# keeps the RHS of the field that LEAVES it and takes the RHS of the field that ENTERS it from its neighbour, i.e. (A.16) with
# the zeroed incoming part replaced by the neighbour's; the zero-speed fields (psi, tangential Phi) keep their own RHS.
def wave_rhs_raw(u, Nr, Nt, Np, rmin, rmax):
    """(-Pi, -d_i Phi_i, -d_x Pi, -d_y Pi, -d_z Pi) on one shell from the oracle gradient, no boundary treatment."""
    u, nf = _state(u, Nr, Nt, Np)
    assert nf == 5
    u = u.reshape(5, Np, Nt, Nr)
    g = gradient(u[1:], Nr, Nt, Np, rmin, rmax)                  # [3, 4 (Pi, Phi_x, Phi_y, Phi_z), Np, Nt, Nr]
    return np.stack([-u[1], -(g[0, 1] + g[1, 2] + g[2, 3]), -g[0, 0], -g[1, 0], -g[2, 0]])


def _unit_normal(Nt, Np):
    th = np.pi * (np.arange(Nt) + 0.5) / Nt
    ph = 2.0 * np.pi * np.arange(Np) / Np
    PH, TH = np.meshgrid(ph, th, indexing="ij")
    return np.stack([np.sin(TH) * np.cos(PH), np.sin(TH) * np.sin(PH), np.cos(TH)])      # [3, Np, Nt]


def nested_wave_rhs(us, shells):
    """us[a]: state [5, Np, Nt, Nr_a] of shell a; shells[a] = dict(Nr, Nt, Np, rmin, rmax), shells[a]['rmax'] == shells[a+1]['rmin'].
    Freezing condition (A.16) on the innermost and outermost sphere, characteristic exchange on every interface."""
    n = _unit_normal(shells[0]["Nt"], shells[0]["Np"])
    raw = [wave_rhs_raw(u, s["Nr"], s["Nt"], s["Np"], s["rmin"], s["rmax"]) for u, s in zip(us, shells)]
    out = [r.copy() for r in raw]

    def put(d, k, dPi, ndPhi, own):
        """row k of d: Pi-RHS dPi, normal part of the Phi-RHS ndPhi, tangential part and psi from `own`"""
        tang = own[2:5, ..., k] - n * np.sum(n * own[2:5, ..., k], axis=0)
        d[1, ..., k] = dPi
        d[2:5, ..., k] = tang + n * ndPhi

    for a in range(len(shells) - 1):
        assert shells[a]["rmax"] == shells[a + 1]["rmin"] and shells[a]["Nt"] == shells[a + 1]["Nt"]
        A, B = raw[a], raw[a + 1]
        Up = A[1, ..., -1] + np.sum(n * A[2:5, ..., -1], axis=0)     # leaves shell a outward, enters shell a+1
        Um = B[1, ..., 0] - np.sum(n * B[2:5, ..., 0], axis=0)       # leaves shell a+1 inward, enters shell a
        put(out[a], -1, 0.5 * (Up + Um), 0.5 * (Up - Um), A)
        put(out[a + 1], 0, 0.5 * (Up + Um), 0.5 * (Up - Um), B)
    first, last = raw[0], raw[-1]
    Um = first[1, ..., 0] - np.sum(n * first[2:5, ..., 0], axis=0)   # inner physical boundary: the outward-moving U^+ enters: frozen
    put(out[0], 0, 0.5 * Um, -0.5 * Um, first)
    Up = last[1, ..., -1] + np.sum(n * last[2:5, ..., -1], axis=0)   # outer physical boundary: the inward-moving U^- enters: frozen
    put(out[-1], -1, 0.5 * Up, 0.5 * Up, last)
    return out


def nested_wave_dt(shells, lam=4.0):
    return min(wave_dt(s["Nr"], s["Nt"], s["Np"], s["rmin"], s["rmax"], lam) for s in shells)


def nested_wave_rk4(us, shells, L, tensors, dt, nsteps):
    """Classical RK4 of the coupled shells, Yn filter per shell at the places of wave_rk4 (reading W5)."""
    F = lambda vs: [tensor_filter(v, s["Nr"], s["Nt"], s["Np"], L, tensors) for v, s in zip(vs, shells)]
    R = lambda vs: nested_wave_rhs(vs, shells)
    ax = lambda vs, c, ks: [v + c * k for v, k in zip(vs, ks)]
    us = F([np.array(u, dtype=np.float64) for u in us])
    for _ in range(nsteps):
        k1 = R(us)
        k2 = R(F(ax(us, 0.5 * dt, k1)))
        k3 = R(F(ax(us, 0.5 * dt, k2)))
        k4 = R(F(ax(us, dt, k3)))
        us = F([u + dt / 6.0 * (a + 2.0 * b + 2.0 * c + d) for u, a, b, c, d in zip(us, k1, k2, k3, k4)])
    return us
