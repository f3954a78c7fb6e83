"""Pins for the oracle's filter matrices, spin-n sphere filter and Yn tensor filter (O8-O12).

Routes independent of the oracle's Householder QR / its tensor loop: numpy's SVD pseudo-inverse,
the Moore-Penrose axioms, closed-form truncation of synthetic expansions, eq. (50), App. B (B.3),
the rank+degree rule of PAPER.md:438-440, and eq. (60) assembled by hand for a vector.
"""
import numpy as np
import pytest

import oracle


def _Y(n, l, m, N):
    """Y^n_lm on the N x 2N grid, array [j, i] complex (eq. 46)."""
    th = np.pi * (np.arange(N) + 0.5) / N
    ph = 2 * np.pi * np.arange(2 * N) / (2 * N)
    P = np.array([oracle.spin_P(n, m, l, t)[l] for t in th])
    return np.exp(1j * m * ph)[:, None] * P[None, :]


@pytest.mark.parametrize("N,L", [(8, 6), (12, 7), (24, 19)])
def test_filter_matrix_vs_numpy_svd(N, L):
    """eq. 62 with eq. 49: F = P f P^+, P^+ by numpy's SVD (the paper's route)."""
    for n in range(-3, 4):
        for m in range(-(N - 1), N):
            F = oracle.filter_matrix(N, L, n, m)
            l0 = max(abs(n), abs(m))
            if l0 > L:
                assert np.all(F == 0)
                continue
            P = oracle.synthesis_matrix(N, n, m)
            assert P.shape == (N, N - l0)
            Pp = np.linalg.pinv(P)
            f = np.array([1.0 if l0 + q <= L else 0.0 for q in range(N - l0)])
            assert np.max(np.abs(F - (P * f) @ Pp)) < 5e-14
            # Moore-Penrose axioms for the full projector and facts of 8(c)
            Ffull = oracle.filter_matrix(N, N - 1, n, m)
            assert np.max(np.abs(Ffull @ P - P)) < 5e-14
            assert np.max(np.abs(Ffull - Ffull.T)) < 5e-14
            assert np.max(np.abs(F @ F - F)) < 5e-14
            assert np.linalg.matrix_rank(F, tol=1e-9) == L - l0 + 1
            # F^n_{-m} = F^{-n}_m (eq. 47)
            assert np.max(np.abs(oracle.filter_matrix(N, L, n, -m) - oracle.filter_matrix(N, L, -n, m))) < 5e-14


def test_filter_matrix_large_N_conditioning():
    """N = 96 (config 4): QR route against numpy SVD on a few (n, m); cond(P) stays small (Q14)."""
    N, L = 96, 91
    for n, m in [(0, 0), (3, 0), (-3, 1), (2, 40), (1, 90), (-1, -91)]:
        P = oracle.synthesis_matrix(N, n, m)
        assert np.linalg.cond(P) < 20
        l0 = max(abs(n), abs(m))
        f = np.array([1.0 if l0 + q <= L else 0.0 for q in range(N - l0)])
        F = oracle.filter_matrix(N, L, n, m)
        assert np.max(np.abs(F - (P * f) @ np.linalg.pinv(P))) < 2e-13


@pytest.mark.parametrize("n", [0, 1, -1, 2, -3])
def test_sphere_filter_truncates_exactly(n):
    """O10: an expansion in grid harmonics is truncated to its l <= L part exactly (reading Q11(i));
    pure modes L < l <= N-1 are annihilated; the Nyquist column cos(N phi) is dropped (Q5)."""
    N, L = 12, 8
    rng = np.random.default_rng(3 + n)
    g = np.zeros((2 * N, N), complex); keep = np.zeros_like(g)
    for l in range(abs(n), N):
        for m in range(-l, l + 1):
            c = rng.standard_normal() + 1j * rng.standard_normal()
            Y = _Y(n, l, m, N)
            g += c * Y
            if l <= L:
                keep += c * Y
    out = oracle.spin_filter_sphere(N, L, n, g)
    assert np.max(np.abs(out - keep)) < 2e-13
    for l in range(L + 1, N):
        Y = _Y(n, l, min(l, 2), N)
        assert np.max(np.abs(oracle.spin_filter_sphere(N, L, n, Y))) < 2e-14
    ph = 2 * np.pi * np.arange(2 * N) / (2 * N)
    nyq = np.cos(N * ph)[:, None] * np.ones((1, N))
    assert np.max(np.abs(oracle.spin_filter_sphere(N, N - 1, n, nyq))) < 1e-14


def test_sphere_filter_conjugation_eq50_and_wrong_spin():
    """eq. 50: conj(F_n f) = F_{-n}(conj f); and F_n f != F_{-n} f for n != 0."""
    N, L = 10, 7
    rng = np.random.default_rng(11)
    g = rng.standard_normal((2 * N, N)) + 1j * rng.standard_normal((2 * N, N))
    for n in (1, 2, 3):
        a = oracle.spin_filter_sphere(N, L, n, g)
        b = oracle.spin_filter_sphere(N, L, -n, np.conj(g))
        assert np.max(np.abs(np.conj(a) - b)) < 1e-14
        assert np.max(np.abs(a - oracle.spin_filter_sphere(N, L, -n, g))) > 1e-2


def test_B3_mx_is_two_spin1_modes():
    """PAPER.md:771-778 (B.3): m_x = (cos th cos ph - i sin ph)/sqrt 2 = sqrt(2 pi/3)(Y^1_11 - Y^1_1,-1):
    preserved by F_{+1} even at L = 1, not by F_0 or F_{-1}.  Pins the sign pairing (reading Q7)."""
    N = 8
    th = np.pi * (np.arange(N) + 0.5) / N
    ph = 2 * np.pi * np.arange(2 * N) / (2 * N)
    mx = (np.cos(th)[None, :] * np.cos(ph)[:, None] - 1j * np.sin(ph)[:, None] * np.ones((1, N))) / np.sqrt(2)
    two = np.sqrt(2 * np.pi / 3) * (_Y(1, 1, 1, N) - _Y(1, 1, -1, N))
    assert np.max(np.abs(mx - two)) < 1e-15
    assert np.max(np.abs(oracle.spin_filter_sphere(N, 1, 1, mx) - mx)) < 1e-15
    assert np.max(np.abs(oracle.spin_filter_sphere(N, 3, -1, mx) - mx)) > 0.05
    assert np.max(np.abs(oracle.spin_filter_sphere(N, 3, 0, mx) - mx)) > 0.05
    # the analysis coefficients of the m = +1 Fourier column: exactly one entry sqrt(2 pi/3) at l = 1
    c = oracle.spin_analysis(N, 1, 1, (np.sqrt(2 * np.pi / 3) * _Y(1, 1, 1, N))[0, :].real)
    assert abs(c[0] - np.sqrt(2 * np.pi / 3)) < 1e-14 and np.max(np.abs(c[1:])) < 1e-14


def _unit_vectors(N, Nr=1):
    th = np.pi * (np.arange(N) + 0.5) / N
    ph = 2 * np.pi * np.arange(2 * N) / (2 * N)
    T, P = np.meshgrid(th, ph, indexing="xy")       # [j, i]
    nx, ny, nz = np.sin(T) * np.cos(P), np.sin(T) * np.sin(P), np.cos(T)
    rep = lambda a: np.repeat(a[:, :, None], Nr, axis=2)
    return rep(nx), rep(ny), rep(nz)


def _rand_poly(rng, nx, ny, nz, p):
    f = np.zeros_like(nx)
    for a in range(p + 1):
        for b in range(p + 1 - a):
            f += rng.standard_normal() * nx ** a * ny ** b * nz ** (p - a - b)
    return f


TENS = {
    0: {"rank": 0, "dims": (), "sym": (-1, -1)},
    1: {"rank": 1, "dims": (3,), "sym": (-1, -1)},
    "1t": {"rank": 1, "dims": (4,), "sym": (-1, -1)},
    2: {"rank": 2, "dims": (4, 4), "sym": (0, 1)},
    "2g": {"rank": 2, "dims": (3, 3), "sym": (-1, -1)},
    3: {"rank": 3, "dims": (3, 4, 4), "sym": (1, 2)},
}


@pytest.mark.parametrize("key,nsp", [(0, 0), (1, 1), ("1t", 1), (2, 2), ("2g", 2), (3, 3)])
def test_tensor_filter_rank_plus_degree_rule(key, nsp):
    """PAPER.md:438-440 (T10): components that are degree-p polynomials in the unit vector are
    preserved iff p + (number of spatial indices) <= L.  Also idempotence and radius selection."""
    N, L, Nr = 12, 7, 2
    t = dict(TENS[key])
    nc = oracle.ncomp(t["rank"], t["dims"], t["sym"])
    t["fields"] = list(range(nc))
    nx, ny, nz = _unit_vectors(N, Nr)
    rng = np.random.default_rng(17)
    p_ok = L - nsp
    u = np.stack([_rand_poly(rng, nx, ny, nz, p_ok) for _ in range(nc)])
    out = oracle.tensor_filter(u, Nr, N, 2 * N, L, [t])
    assert np.max(np.abs(out - u)) < 1e-13 * np.max(np.abs(u))
    u2 = np.stack([_rand_poly(rng, nx, ny, nz, p_ok + 1) for _ in range(nc)])
    out2 = oracle.tensor_filter(u2, Nr, N, 2 * N, L, [t])
    assert np.max(np.abs(out2 - u2)) > 1e-4 * np.max(np.abs(u2))
    assert np.max(np.abs(oracle.tensor_filter(out2, Nr, N, 2 * N, L, [t]) - out2)) < 1e-13 * np.max(np.abs(u2))
    # untouched fields / radii: ksel filters one radius only
    outk = oracle.tensor_filter(u2, Nr, N, 2 * N, L, [t], ksel=1)
    assert np.all(outk[..., 0] == u2[..., 0]) and np.all(outk[..., 1] == out2[..., 1])


def test_tensor_filter_vector_equals_eq60_by_hand():
    """eq. (54)-(56), (60) assembled in numpy from the sphere filter: v_r = r.v -> F_0,
    m.v -> F_{+1} (reading Q7), recombined with the conjugate dyad; t component -> F_0 (Q17)."""
    N, L = 10, 6
    rng = np.random.default_rng(23)
    u = rng.standard_normal((4, 2 * N, N, 1))
    t = {"rank": 1, "dims": (4,), "sym": (-1, -1), "fields": [0, 1, 2, 3]}
    got = oracle.tensor_filter(u, 1, N, 2 * N, L, [t])
    nx, ny, nz = [a[:, :, 0] for a in _unit_vectors(N)]
    th = np.pi * (np.arange(N) + 0.5) / N
    ph = 2 * np.pi * np.arange(2 * N) / (2 * N)
    T, P = np.meshgrid(th, ph, indexing="xy")
    rh = np.stack([nx, ny, nz])
    tha = np.stack([np.cos(T) * np.cos(P), np.cos(T) * np.sin(P), -np.sin(T)])
    pha = np.stack([-np.sin(P), np.cos(P), np.zeros_like(P)])
    mv = (tha + 1j * pha) / np.sqrt(2)
    v = u[1:, :, :, 0]
    vr = oracle.spin_filter_sphere(N, L, 0, np.sum(rh * v, axis=0))
    vm = oracle.spin_filter_sphere(N, L, 1, np.sum(mv * v, axis=0))
    want = rh * vr.real + 2 * np.real(vm[None] * np.conj(mv))     # (m.v) mbar + c.c.
    assert np.max(np.abs(got[1:, :, :, 0] - want)) < 2e-14
    want_t = oracle.spin_filter_sphere(N, L, 0, u[0, :, :, 0]).real
    assert np.max(np.abs(got[0, :, :, 0] - want_t)) < 2e-14


def test_tensor_filter_rank2_synthesised_in_spin_space():
    """A symmetric spatial rank-2 tensor built as T = Re-part of sum_e T~_e conj(E)conj(E) with
    T~_mm = sum c_lm Y^{+2}_lm, T~_rm = sum Y^{+1}, T~_rr, T~_mmbar = sum Y^0: the Yn filter must
    return the same construction with every expansion cut at l <= L (closed-form truncation)."""
    N, L = 12, 8
    rng = np.random.default_rng(29)
    th = np.pi * (np.arange(N) + 0.5) / N
    ph = 2 * np.pi * np.arange(2 * N) / (2 * N)
    T, P = np.meshgrid(th, ph, indexing="xy")
    rh = np.stack([np.sin(T) * np.cos(P), np.sin(T) * np.sin(P), np.cos(T)]).astype(complex)
    mv = (np.stack([np.cos(T) * np.cos(P), np.cos(T) * np.sin(P), -np.sin(T)]) + 1j * np.stack([-np.sin(P), np.cos(P), 0 * P])) / np.sqrt(2)

    def expand(n, real):
        full = np.zeros((2 * N, N), complex); cut = np.zeros_like(full)
        for l in range(abs(n), N):
            for m in range(-l, l + 1):
                c = rng.standard_normal() + 1j * rng.standard_normal()
                Y = _Y(n, l, m, N)
                full += c * Y
                if l <= L:
                    cut += c * Y
        if real:       # a real spin-0 function: add the conjugate
            full, cut = full + np.conj(full), cut + np.conj(cut)
        return full, cut

    comps = {"mm": expand(2, False), "rm": expand(1, False), "rr": expand(0, True), "mmb": expand(0, True)}

    def build(which):
        g = {k: v[which] for k, v in comps.items()}
        Tab = np.zeros((3, 3, 2 * N, N), complex)
        mb = np.conj(mv)
        for a in range(3):
            for b in range(3):
                # T^{ab} = T~_e conj(E_1)^a conj(E_2)^b summed over e, T symmetric and real
                Tab[a, b] = (g["rr"] * rh[a] * rh[b]
                             + g["mm"] * mb[a] * mb[b] + np.conj(g["mm"]) * mv[a] * mv[b]
                             + g["rm"] * (rh[a] * mb[b] + mb[a] * rh[b]) + np.conj(g["rm"]) * (rh[a] * mv[b] + mv[a] * rh[b])
                             + g["mmb"] * (mv[a] * mb[b] + mb[a] * mv[b]))
        assert np.max(np.abs(Tab.imag)) < 1e-13
        return Tab.real

    Tf, Tc = build(0), build(1)
    idx = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
    u = np.stack([Tf[a, b] for a, b in idx])[..., None]
    want = np.stack([Tc[a, b] for a, b in idx])[..., None]
    t = {"rank": 2, "dims": (3, 3), "sym": (0, 1), "fields": list(range(6))}
    got = oracle.tensor_filter(u, 1, N, 2 * N, L, [t])
    assert np.max(np.abs(got - want)) < 5e-13 * np.max(np.abs(u))
    assert np.max(np.abs(u - want)) > 1e-2          # the cut removed something
    scal = [{"rank": 0, "dims": (), "sym": (-1, -1), "fields": [c]} for c in range(6)]
    assert np.max(np.abs(oracle.tensor_filter(u, 1, N, 2 * N, L, scal) - want)) > 1e-2   # Y-filter differs
