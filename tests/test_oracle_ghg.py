"""Pins of the GHG right-hand-side oracle (oracle/ghg_oracle.c; Appendix A) against what the paper and the
mathematics fix, none of them the oracle's own formulas retyped:
  * the Kerr-Schild metric (A.17) is a static solution of the vacuum Einstein equations, so the RHS (A.8)-(A.10) of data
    built from it must vanish up to the truncation error of the spectral derivatives and fall exponentially with the
    resolution ("rhs -> round-off for static data"); a dropped term, a wrong sign or a misplaced index
    leaves an O(1) residual that does not converge.  Checked for the centred hole and for a displaced one (no symmetry);
  * Minkowski: exactly zero;
  * lapse, shift, inverse 3-metric against the closed forms (A.19);
  * boundary condition (A.20)-(A.21): the incoming characteristic fields of (A.14) are frozen, the outgoing one and
    d_t g_ab keep the value of the unconstrained RHS.
"""
import numpy as np

import oracle
import synth

RMIN, RMAX = 1.8, 6.8


def _static_residual(Nr, Nt, center, bc=False):
    Np = 2 * Nt
    g = synth.kerr_schild_metric(Nr, Nt, Np, RMIN, RMAX, center=center)
    u, H, dH = oracle.ghg_init(g, Nr, Nt, Np, RMIN, RMAX)
    du = oracle.gradient(u, Nr, Nt, Np, RMIN, RMAX)
    rhs = oracle.ghg_rhs(u, du, H, dH, Nr, Nt, Np, RMIN, RMAX, bc_outer=bc)
    return [float(np.abs(rhs[a:b]).max()) for a, b in ((0, 10), (10, 20), (20, 50))]


def test_kerr_schild_is_static_centred_hole_converges_exponentially():
    res = {Nr: _static_residual(Nr, 8, (0.0, 0.0, 0.0)) for Nr in (9, 13, 17, 25)}
    for Nr in res:
        assert res[Nr][0] < 1e-15                       # (A.8) vanishes identically by the construction of k_ab
    for a, b in ((9, 13), (13, 17), (17, 25)):
        assert res[b][1] < 0.1 * res[a][1] and res[b][2] < 0.1 * res[a][2]
    assert res[9][1] < 0.1                               # already small at 9 radial points ...
    assert res[25][1] < 1e-7 and res[25][2] < 1e-8       # ... and at truncation level at 25


def test_kerr_schild_is_static_displaced_hole_converges_in_r_and_angle():
    c = (0.15, -0.1, 0.12)
    coarse, fine_r, fine = _static_residual(11, 6, c), _static_residual(21, 6, c), _static_residual(21, 12, c)
    assert fine[1] < 1e-5 and fine[2] < 1e-6
    assert fine[1] < 0.05 * coarse[1] and fine[2] < 0.05 * coarse[2]
    assert fine[1] < 0.1 * fine_r[1]                     # at Ntheta = 6 the angular error dominates; 12 removes it


def test_static_residual_with_boundary_condition_still_converges():
    a, b = _static_residual(13, 8, (0.0, 0.0, 0.0), bc=True), _static_residual(25, 8, (0.0, 0.0, 0.0), bc=True)
    assert b[1] < 1e-7 and b[1] < 1e-3 * a[1]


def test_minkowski_gives_zero():
    Nr, Nt, Np = 7, 6, 12
    g = synth.minkowski_metric(Nr, Nt, Np)
    u, H, dH = oracle.ghg_init(g, Nr, Nt, Np, 1.0, 3.0)
    assert np.abs(u[10:]).max() < 1e-13 and np.abs(H).max() < 1e-13
    u[10:] = 0.0
    z = np.zeros((3, 50, Np, Nt, Nr))
    rhs = oracle.ghg_rhs(u, z, np.zeros_like(H), np.zeros_like(dH), Nr, Nt, Np, 1.0, 3.0)
    assert np.abs(rhs).max() == 0.0


def test_lapse_shift_inverse_metric_closed_forms_A19():
    Nr, Nt, Np = 9, 6, 12
    g = synth.kerr_schild_metric(Nr, Nt, Np, RMIN, RMAX)
    u = np.zeros((50, Np, Nt, Nr)); u[:10] = g
    out = oracle.ghg_lapse_shift(u, Nr, Nt, Np)
    x, y, z = synth.grid_xyz(Nr, Nt, Np, RMIN, RMAX)
    r = np.sqrt(x * x + y * y + z * z)
    f = 2.0 / r
    l = [x / r, y / r, z / r]
    assert np.abs(out[0] - 1.0 / np.sqrt(1.0 + f)).max() < 1e-15
    for i in range(3):
        assert np.abs(out[1 + i] - l[i] * f / (1.0 + f)).max() < 1e-15
    c = 4
    for i in range(3):
        for j in range(i, 3):
            assert np.abs(out[c] - ((i == j) - f / (1.0 + f) * l[i] * l[j])).max() < 1e-15
            c += 1


def test_boundary_condition_freezes_incoming_characteristic_fields():
    """(A.14): e^1 = -g + k + s^i d_i (speed alpha - b, outgoing at the outer boundary), e^2 = -g + k - s^i d_i and the two
    tangential combinations of d_i (incoming).  With (A.20)-(A.21): d_t e^2 = 0, tangential d_t d = 0, d_t e^1 and d_t g
    unchanged.  s_i is rebuilt here with numpy from the state's own 3-metric."""
    Nr, Nt, Np = 9, 6, 12
    g = synth.kerr_schild_metric(Nr, Nt, Np, RMIN, RMAX, center=(0.1, 0.05, -0.08))
    u, H, dH = oracle.ghg_init(g, Nr, Nt, Np, RMIN, RMAX)
    u = synth.perturbed_ghg_state(u, 1e-2, 7)
    du = oracle.gradient(u, Nr, Nt, Np, RMIN, RMAX)
    free = oracle.ghg_rhs(u, du, H, dH, Nr, Nt, Np, RMIN, RMAX, bc_outer=False)
    bc = oracle.ghg_rhs(u, du, H, dH, Nr, Nt, Np, RMIN, RMAX, bc_outer=True)
    assert np.array_equal(free[..., :Nr - 1], bc[..., :Nr - 1])            # interior untouched
    x, y, z = synth.grid_xyz(Nr, Nt, Np, RMIN, RMAX)
    sym = [[0, 1, 2, 3], [1, 4, 5, 6], [2, 5, 7, 8], [3, 6, 8, 9]]
    worst = 0.0
    for j in range(Np):
        for i in range(Nt):
            k = Nr - 1
            gam = np.array([[u[sym[a + 1][b + 1], j, i, k] for b in range(3)] for a in range(3)])
            gi = np.linalg.inv(gam)
            l = np.array([x[j, i, k], y[j, i, k], z[j, i, k]]); l /= np.linalg.norm(l)
            s_dn = l / np.sqrt(l @ gi @ l)
            s_up = gi @ s_dn
            for ab in range(10):
                tg0, tk0, td0 = free[ab, j, i, k], free[10 + ab, j, i, k], np.array([free[20 + 10 * q + ab, j, i, k] for q in range(3)])
                tg1, tk1, td1 = bc[ab, j, i, k], bc[10 + ab, j, i, k], np.array([bc[20 + 10 * q + ab, j, i, k] for q in range(3)])
                scale = max(abs(tg0), abs(tk0), np.abs(td0).max(), 1e-30)
                worst = max(worst, abs(tg1 - tg0) / scale)
                worst = max(worst, abs((-tg1 + tk1 - s_up @ td1)) / scale)                       # incoming e^2 frozen
                worst = max(worst, np.abs(td1 - s_dn * (s_up @ td1)).max() / scale)              # tangential part frozen
                worst = max(worst, abs((-tg1 + tk1 + s_up @ td1) - (-tg0 + tk0 + s_up @ td0)) / scale)   # outgoing kept
    assert worst < 1e-13


def test_characteristic_speeds_printed_in_the_paper():
    """"in the numerical example r_min = 1.80, and the eigenvalues range from -1.45 ...  For r_min = 2.00, the
    fastest eigenspeed is -sqrt(2) = -1.41, for r_min = 1.50 it is -1.53" -- the speed -alpha - b of (A.14) with b = s_k beta^k
    and s_i the unit normal w.r.t. gamma^{ij}, all taken from the oracle's 3+1 split of the Kerr-Schild data."""
    for rmin, printed in ((1.80, -1.45), (2.00, -1.41), (1.50, -1.53)):
        Nr, Nt, Np = 5, 4, 8
        g = synth.kerr_schild_metric(Nr, Nt, Np, rmin, rmin + 5.0)
        u = np.zeros((50, Np, Nt, Nr)); u[:10] = g
        out = oracle.ghg_lapse_shift(u, Nr, Nt, Np)
        x, y, z = synth.grid_xyz(Nr, Nt, Np, rmin, rmin + 5.0)
        j, i, k = 3, 1, 0                                          # a point on the inner boundary
        l = np.array([x[j, i, k], y[j, i, k], z[j, i, k]]); l /= np.linalg.norm(l)
        gi = np.zeros((3, 3)); c = 4
        for a in range(3):
            for b in range(a, 3):
                gi[a, b] = gi[b, a] = out[c, j, i, k]; c += 1
        s_dn = l / np.sqrt(l @ gi @ l)
        alpha, beta_up = out[0, j, i, k], out[1:4, j, i, k]
        v = -alpha - s_dn @ beta_up
        assert abs(v - printed) < 0.006, (rmin, v)
        assert abs((alpha - s_dn @ beta_up)) < 1e-12 if rmin == 2.00 else True      # the outgoing speed vanishes on the horizon


# ---- the terms proportional to the constraints C_iab = d_i g_ab - d_iab and C_a = H_a + Gamma_a --------------------------
# They vanish identically on the constraint-satisfying static data above, so they get their own pins: the LINEAR RESPONSE of
# the printed equations (A.9), (A.10) on a flat background to ONE small perturbation at a time has a closed form.  The
# response is taken by a central difference in eps (even orders cancel), the oracle receives the "numerical derivatives" du
# as an argument, so every derivative slot can be driven independently.  Backgrounds: Minkowski (alpha = 1, beta = 0,
# n^a = (1,0,0,0), n_a = (-1,0,0,0)) and Minkowski in Galilean-shifted coordinates x' = x + b t (a constant metric
# g_tt = -1 + b.b, g_ti = b_i, g_ij = delta_ij: alpha = 1, beta^i = b_i, gamma^ij = delta^ij, Gamma = 0).
_SYM = [[0, 1, 2, 3], [1, 4, 5, 6], [2, 5, 7, 8], [3, 6, 8, 9]]
_G = (3, 2, 4)            # Nr, Nt, Np: the RHS is pointwise


def _flat_state(b=(0.0, 0.0, 0.0)):
    Nr, Nt, Np = _G
    b = np.asarray(b, dtype=float)
    g4 = np.diag([-1.0, 1.0, 1.0, 1.0])
    g4[0, 0] += b @ b
    g4[0, 1:] = g4[1:, 0] = b
    u = np.zeros((50, Np, Nt, Nr))
    for a in range(4):
        for c in range(a, 4):
            u[_SYM[a][c]] = g4[a, c]
    return u, g4


def _sym_field(rng, lead=()):
    """random [*lead, 4, 4, Np, Nt, Nr], symmetric in the two 4-indices"""
    Nr, Nt, Np = _G
    s = rng.standard_normal(tuple(lead) + (4, 4, Np, Nt, Nr))
    return s + np.swapaxes(s, len(lead), len(lead) + 1)


def _response(make, eps=1e-6):
    """(rhs(+eps) - rhs(-eps)) / (2 eps) of oracle.ghg_rhs; make(eps) -> (u, du, H, dH).  Returns tg [4,4,..], tk, td [3,4,4,..]."""
    Nr, Nt, Np = _G
    r = [oracle.ghg_rhs(*make(e), Nr, Nt, Np, 1.0, 2.0) for e in (eps, -eps)]
    d = (r[0] - r[1]) / (2 * eps)
    full = lambda base: np.array([[d[base + _SYM[a][c]] for c in range(4)] for a in range(4)])
    return full(0), full(10), np.array([full(20 + 10 * i) for i in range(3)])


def _put(u, base, s):
    for a in range(4):
        for c in range(a, 4):
            u[base + _SYM[a][c]] += s[a, c]


def test_A9_minus_alpha_d_iab_term():
    """Minkowski, d_iab = eps c_iab, everything else zero: (A.9) reduces to d_t d_iab = -eps c_iab (the -alpha d_iab term;
    the n n d k and gamma n d d terms are second order, every derivative slot is zero)."""
    rng = np.random.default_rng(21)
    c = _sym_field(rng, (3,))
    Nr, Nt, Np = _G

    def make(e):
        u, _ = _flat_state()
        for i in range(3):
            _put(u, 20 + 10 * i, e * c[i])
        return u, np.zeros((3, 50, Np, Nt, Nr)), np.zeros((4, Np, Nt, Nr)), np.zeros((3, 4, Np, Nt, Nr))

    tg, tk, td = _response(make)
    assert np.abs(td + c).max() < 1e-8
    assert np.abs(tg).max() < 1e-8                      # (A.8): beta = 0, k = 0


def test_A9_plus_alpha_di_g_ab_term():
    """Minkowski + eps h_ab with the derivative slot of g_ab driven by eps s_iab, d = k = 0: (A.9) gives d_t d_iab = +eps s_iab
    (the +alpha d_i g_ab term) and (A.10) nothing at first order (its -beta^k d_k g_ab is second order here)."""
    rng = np.random.default_rng(22)
    h, s = _sym_field(rng), _sym_field(rng, (3,))
    Nr, Nt, Np = _G

    def make(e):
        u, _ = _flat_state()
        _put(u, 0, e * h)
        du = np.zeros((3, 50, Np, Nt, Nr))
        for i in range(3):
            _put(du[i], 0, e * s[i])
        return u, du, np.zeros((4, Np, Nt, Nr)), np.zeros((3, 4, Np, Nt, Nr))

    tg, tk, td = _response(make)
    assert np.abs(td - s).max() < 1e-8
    assert np.abs(tk).max() < 1e-8


def test_A10_gamma0_constraint_damping_term():
    """Minkowski, H_a = eps w_a (no derivative), everything else zero: Gamma_a = 0, nabla_(a H_b) = 0 at first order, so (A.10)
    reduces to d_t k_ab = gamma0 alpha (2 delta^c_(a n_b) - g_ab n^c)(H_c + Gamma_c) = eps (n_b w_a + n_a w_b - eta_ab n^c w_c)
    with n_a = (-1,0,0,0), n^a = (1,0,0,0), gamma0 = 1."""
    rng = np.random.default_rng(23)
    Nr, Nt, Np = _G
    w = rng.standard_normal((4, Np, Nt, Nr))
    eta = np.diag([-1.0, 1.0, 1.0, 1.0])
    n_dn, n_up = np.array([-1.0, 0, 0, 0]), np.array([1.0, 0, 0, 0])

    def make(e):
        u, _ = _flat_state()
        return u, np.zeros((3, 50, Np, Nt, Nr)), e * w, np.zeros((3, 4, Np, Nt, Nr))

    tg, tk, td = _response(make)
    nw = np.einsum("c,c...->...", n_up, w)
    want = np.einsum("b,a...->ab...", n_dn, w) + np.einsum("a,b...->ab...", n_dn, w) - eta[:, :, None, None, None] * nw
    assert np.abs(tk - want).max() < 1e-8
    assert np.abs(td).max() < 1e-8 and np.abs(tg).max() < 1e-8


def test_A10_minus_beta_dk_g_ab_term():
    """Shifted flat background (beta^i = b_i), derivative slot of g_ab driven by eps s_kab, d = k = 0: the only first-order
    terms are d_t d_iab = alpha s_iab and, in (A.10), -beta^k d_k g_ab = -eps b^k s_kab."""
    rng = np.random.default_rng(24)
    b = np.array([0.3, -0.2, 0.25])
    s = _sym_field(rng, (3,))
    Nr, Nt, Np = _G

    def make(e):
        u, _ = _flat_state(b)
        du = np.zeros((3, 50, Np, Nt, Nr))
        for i in range(3):
            _put(du[i], 0, e * s[i])
        return u, du, np.zeros((4, Np, Nt, Nr)), np.zeros((3, 4, Np, Nt, Nr))

    tg, tk, td = _response(make)
    assert np.abs(tk + np.einsum("k,k...->...", b, s)).max() < 1e-8
    assert np.abs(td - s).max() < 1e-8


def test_A10_plus_beta_d_iab_term_and_A8():
    """Shifted flat background, d_iab = eps v_i w_ab with w_ab trace-free and orthogonal to V_a = (b.v, v_i) (built with numpy
    from the constant 4-metric): then D_a g_bc = eps V_a w_bc gives Gamma_c = eps (V^b w_bc - V_c tr w / 2) = 0, so the
    constraint-damping term is silent and (A.10) reduces to its last term, d_t k_ab = +beta^i d_iab = eps (b.v) w_ab;
    (A.8) gives the same for d_t g_ab, (A.9) gives -alpha d_iab."""
    rng = np.random.default_rng(25)
    b = np.array([0.3, -0.2, 0.25])
    v = np.array([0.7, 0.4, -0.5])
    _, g4 = _flat_state(b)
    gi = np.linalg.inv(g4)
    V_dn = np.concatenate([[b @ v], v])
    V_up = gi @ V_dn
    VV = V_dn @ V_up
    assert abs(VV) > 0.1
    Pi = np.eye(4) - np.outer(V_up, V_dn) / VV                  # Pi^c_a: projects orthogonally to V
    S = rng.standard_normal((4, 4)); S = S + S.T
    w = Pi.T @ S @ Pi
    hproj = g4 - np.outer(V_dn, V_dn) / VV
    w = w - np.einsum("ab,ab->", gi, w) / 3.0 * hproj
    assert np.abs(w @ V_up).max() < 1e-13 and abs(np.einsum("ab,ab->", gi, w)) < 1e-13 and np.abs(w).max() > 0.1
    Nr, Nt, Np = _G
    wf = w[:, :, None, None, None] * np.ones((Np, Nt, Nr))

    def make(e):
        u, _ = _flat_state(b)
        for i in range(3):
            _put(u, 20 + 10 * i, e * v[i] * wf)
        return u, np.zeros((3, 50, Np, Nt, Nr)), np.zeros((4, Np, Nt, Nr)), np.zeros((3, 4, Np, Nt, Nr))

    tg, tk, td = _response(make)
    assert np.abs(tk - (b @ v) * wf).max() < 1e-8
    assert np.abs(tg - (b @ v) * wf).max() < 1e-8
    assert np.abs(td + v[:, None, None, None, None, None] * wf[None]).max() < 1e-8
