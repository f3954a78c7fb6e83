/*
 * sp_oracle.c -- CPU ORACLE for the hot path of Bruegmann's CFF pseudospectral matrix
 * method (arXiv:1104.3408): Cartesian gradient by differentiation matrices and the
 * spin-weighted spherical-harmonic (Yn) tensor filter.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA library in
 * paper_1104_3408_b200/ and neither includes the other.
 *
 * Style: plain C, naive loops over the index definitions in the paper's order and
 * notation, every sum accumulated in `long double`, no blocking, fusion or reordering.
 * Matrices are evaluated in long double and rounded ONCE to double (the matrices are
 * the definition of the method: SURVEY.md 8(c) Q18); the products then use these double
 * matrices with long double accumulation.  Citations are PAPER.md:<line> (section/eq.).
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): App. B closed forms, textbook
 * Y_lm / sY_lm for l<=3, the explicit Wigner-d sum, (B.2) inner products, orthonormality,
 * pseudo-inverse axioms against numpy's SVD, exact derivatives of polynomials in x,y,z,
 * filter idempotence / preservation / annihilation, (B.3), rank+degree rule.  Nothing
 * here is "parity unpinned".
 *
 * Layout of every state array (single cover, reading Q4):
 *     p = k + Nr*(i + Nt*(j + Np*mu)),  k radial (fastest), i latitude, j longitude, mu field.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>

typedef long double ld;
static const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;

/* ------------------------------------------------------------------------------------
 * O1  Grid.  PAPER.md:57-66 (eq. 2-4), 76 (eq. 5: Np = 2 Nt).
 *   r_k  = (rmax+rmin)/2 - (rmax-rmin)/2 cos(pi k/(Nr-1))
 *   th_i = pi (i+1/2)/Nt,   ph_j = 2 pi j/Np
 * ---------------------------------------------------------------------------------- */
static ld grid_r(int Nr, double rmin, double rmax, int k) {
    return ((ld)rmax + (ld)rmin) / 2 - ((ld)rmax - (ld)rmin) / 2 * cosl(PI_L * k / (Nr - 1));
}
static ld grid_th(int Nt, int i) { return PI_L * ((ld)i + 0.5L) / Nt; }
static ld grid_ph(int Np, int j) { return 2 * PI_L * j / Np; }

void orc_grid(int Nr, int Nt, int Np, double rmin, double rmax, double *r, double *th, double *ph) {
    for (int k = 0; k < Nr; k++) r[k] = (double)grid_r(Nr, rmin, rmax, k);
    for (int i = 0; i < Nt; i++) th[i] = (double)grid_th(Nt, i);
    for (int j = 0; j < Np; j++) ph[j] = (double)grid_ph(Np, j);
}

/* ------------------------------------------------------------------------------------
 * O2  Chebyshev differentiation matrix on the extrema grid.  PAPER.md:107-112 (eq. 9).
 *   x_i = -cos(pi i/(N-1));  CD_ij = (c_i/c_j)(-1)^{i+j}/(x_i-x_j), i != j,
 *   CD_ii = -sum_{j!=i} CD_ij;  c_0 = c_{N-1} = 2, else 1;  CD^ = 2 CD/(rmax-rmin).
 * D is row-major N x N: D[i*N+j].
 * ---------------------------------------------------------------------------------- */
void orc_cheb_diff(int N, double rmin, double rmax, double *D) {
    ld *x = malloc(sizeof(ld) * N);
    ld *M = malloc(sizeof(ld) * N * N);
    for (int i = 0; i < N; i++) x[i] = -cosl(PI_L * i / (N - 1));
    for (int i = 0; i < N; i++) {
        ld ci = (i == 0 || i == N - 1) ? 2 : 1;
        ld diag = 0;
        for (int j = 0; j < N; j++) {
            if (j == i) continue;
            ld cj = (j == 0 || j == N - 1) ? 2 : 1;
            ld sgn = ((i + j) % 2 == 0) ? 1 : -1;
            M[i * N + j] = (ci / cj) * sgn / (x[i] - x[j]);
            diag -= M[i * N + j];
        }
        M[i * N + i] = diag;
    }
    ld scale = 2 / ((ld)rmax - (ld)rmin);
    for (int p = 0; p < N * N; p++) D[p] = (double)(scale * M[p]);
    free(x); free(M);
}

/* ------------------------------------------------------------------------------------
 * O3  Fourier differentiation matrix, n even, equally spaced periodic grid of spacing
 * 2 pi/n.  PAPER.md:102-105 (eq. 8):  FD_ij = (-1)^{i+j} / (2 tan((x_i-x_j)/2)), FD_ii = 0,
 * with (x_i-x_j)/2 = (i-j) pi/n (the theta stagger cancels in the difference).
 * ---------------------------------------------------------------------------------- */
void orc_fourier_diff(int n, double *D) {
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) {
            if (i == j) { D[i * n + j] = 0; continue; }
            ld sgn = ((i + j) % 2 == 0) ? 1 : -1;
            D[i * n + j] = (double)(sgn / (2 * tanl(PI_L * (i - j) / n)));
        }
}

/* ------------------------------------------------------------------------------------
 * O4/O5  One-directional derivatives of nf fields.  PAPER.md:98-100 (eq. 7), 142-166
 * (eq. 13-19), 72 (double cover).  Naive loops, long double accumulation.
 * ---------------------------------------------------------------------------------- */
#define IDX(k, i, j, mu) ((size_t)(k) + (size_t)Nr * ((size_t)(i) + (size_t)Nt * ((size_t)(j) + (size_t)Np * (size_t)(mu))))

void orc_dr(int Nr, int Nt, int Np, int nf, double rmin, double rmax, const double *u, double *out) {
    double *D = malloc(sizeof(double) * Nr * Nr);
    orc_cheb_diff(Nr, rmin, rmax, D);
#pragma omp parallel for collapse(2) schedule(static)
    for (int mu = 0; mu < nf; mu++)
        for (int j = 0; j < Np; j++)
            for (int i = 0; i < Nt; i++)
                for (int k = 0; k < Nr; k++) {
                    ld s = 0;
                    for (int kk = 0; kk < Nr; kk++) s += (ld)D[k * Nr + kk] * (ld)u[IDX(kk, i, j, mu)];
                    out[IDX(k, i, j, mu)] = (double)s;
                }
    free(D);
}

/* theta: u_ext[i'] = u[i'] for i' < Nt; u_ext[i', j] = u[2Nt-1-i', (j+Nt) mod Np] for i' >= Nt
 * (f(theta,phi) = f(2pi-theta, pi+phi)); rows 0..Nt-1 of FD_{2Nt}. */
void orc_dtheta(int Nr, int Nt, int Np, int nf, const double *u, double *out) {
    int n2 = 2 * Nt;
    double *D = malloc(sizeof(double) * n2 * n2);
    orc_fourier_diff(n2, D);
#pragma omp parallel for collapse(2) schedule(static)
    for (int mu = 0; mu < nf; mu++)
        for (int j = 0; j < Np; j++) {
            double *uext = malloc(sizeof(double) * n2);
            for (int k = 0; k < Nr; k++) {
                for (int ii = 0; ii < n2; ii++)
                    uext[ii] = (ii < Nt) ? u[IDX(k, ii, j, mu)] : u[IDX(k, n2 - 1 - ii, (j + Nt) % Np, mu)];
                for (int i = 0; i < Nt; i++) {
                    ld s = 0;
                    for (int ii = 0; ii < n2; ii++) s += (ld)D[i * n2 + ii] * (ld)uext[ii];
                    out[IDX(k, i, j, mu)] = (double)s;
                }
            }
            free(uext);
        }
    free(D);
}

void orc_dphi(int Nr, int Nt, int Np, int nf, const double *u, double *out) {
    double *D = malloc(sizeof(double) * Np * Np);
    orc_fourier_diff(Np, D);
#pragma omp parallel for collapse(2) schedule(static)
    for (int mu = 0; mu < nf; mu++)
        for (int j = 0; j < Np; j++)
            for (int i = 0; i < Nt; i++)
                for (int k = 0; k < Nr; k++) {
                    ld s = 0;
                    for (int jj = 0; jj < Np; jj++) s += (ld)D[j * Np + jj] * (ld)u[IDX(k, i, jj, mu)];
                    out[IDX(k, i, j, mu)] = (double)s;
                }
    free(D);
}

/* ------------------------------------------------------------------------------------
 * O6  Chain rule, PAPER.md:86-90 (eq. 6); only d(phi)/dx is printed, the rest is the
 * standard inverse Jacobian of spherical coordinates (reading Q15):
 *   d_x = sin th cos ph d_r + (cos th cos ph / r) d_th - (sin ph /(r sin th)) d_ph
 *   d_y = sin th sin ph d_r + (cos th sin ph / r) d_th + (cos ph /(r sin th)) d_ph
 *   d_z = cos th d_r        - (sin th / r) d_th
 * du is [3][nf] state-shaped: du[(c*nf+mu)*Npts + point].
 * ---------------------------------------------------------------------------------- */
void orc_gradient(int Nr, int Nt, int Np, int nf, double rmin, double rmax, const double *u, double *du) {
    size_t npts = (size_t)Nr * Nt * Np, tot = npts * nf;
    double *ur = malloc(sizeof(double) * tot), *ut = malloc(sizeof(double) * tot), *up = malloc(sizeof(double) * tot);
    orc_dr(Nr, Nt, Np, nf, rmin, rmax, u, ur);
    orc_dtheta(Nr, Nt, Np, nf, u, ut);
    orc_dphi(Nr, Nt, Np, nf, u, up);
    for (int mu = 0; mu < nf; mu++)
        for (int j = 0; j < Np; j++)
            for (int i = 0; i < Nt; i++)
                for (int k = 0; k < Nr; k++) {
                    ld r = grid_r(Nr, rmin, rmax, k), th = grid_th(Nt, i), ph = grid_ph(Np, j);
                    ld st = sinl(th), ct = cosl(th), sp = sinl(ph), cp = cosl(ph);
                    size_t p = IDX(k, i, j, mu);
                    ld a = ur[p], b = ut[p], c = up[p];
                    du[(size_t)(0 * nf + mu) * npts + (p - (size_t)mu * npts)] = (double)(st * cp * a + ct * cp / r * b - sp / (r * st) * c);
                    du[(size_t)(1 * nf + mu) * npts + (p - (size_t)mu * npts)] = (double)(st * sp * a + ct * sp / r * b + cp / (r * st) * c);
                    du[(size_t)(2 * nf + mu) * npts + (p - (size_t)mu * npts)] = (double)(ct * a - st / r * b);
                }
    free(ur); free(ut); free(up);
}

/* Gradient at nsamp sampled outputs (for parity at sizes where the full oracle is slow):
 * sample s is (k,i,j,mu) = samp[4s..4s+3]; out[3s+c] = d_c u at that point.  Same
 * definitions as above, evaluated for the one output only. */
void orc_gradient_at(int Nr, int Nt, int Np, int nf, double rmin, double rmax, const double *u,
                     int nsamp, const int *samp, double *out) {
    int n2 = 2 * Nt;
    double *CD = malloc(sizeof(double) * Nr * Nr), *F2 = malloc(sizeof(double) * n2 * n2), *F3 = malloc(sizeof(double) * Np * Np);
    orc_cheb_diff(Nr, rmin, rmax, CD); orc_fourier_diff(n2, F2); orc_fourier_diff(Np, F3);
    (void)nf;
    for (int s = 0; s < nsamp; s++) {
        int k = samp[4 * s], i = samp[4 * s + 1], j = samp[4 * s + 2], mu = samp[4 * s + 3];
        ld a = 0, b = 0, c = 0;
        for (int kk = 0; kk < Nr; kk++) a += (ld)CD[k * Nr + kk] * (ld)u[IDX(kk, i, j, mu)];
        for (int ii = 0; ii < n2; ii++) {
            double ue = (ii < Nt) ? u[IDX(k, ii, j, mu)] : u[IDX(k, n2 - 1 - ii, (j + Nt) % Np, mu)];
            b += (ld)F2[i * n2 + ii] * (ld)ue;
        }
        for (int jj = 0; jj < Np; jj++) c += (ld)F3[j * Np + jj] * (ld)u[IDX(k, i, jj, mu)];
        a = (double)a; b = (double)b; c = (double)c;   /* the three products are double arrays, as in orc_gradient */
        ld r = grid_r(Nr, rmin, rmax, k), th = grid_th(Nt, i), ph = grid_ph(Np, j);
        ld st = sinl(th), ct = cosl(th), sp = sinl(ph), cp = cosl(ph);
        out[3 * s + 0] = (double)(st * cp * a + ct * cp / r * b - sp / (r * st) * c);
        out[3 * s + 1] = (double)(st * sp * a + ct * sp / r * b + cp / (r * st) * c);
        out[3 * s + 2] = (double)(ct * a - st / r * b);
    }
    free(CD); free(F2); free(F3);
}

/* ------------------------------------------------------------------------------------
 * O7  Spin-weighted harmonics.  PAPER.md:352-356 (eq. 46-47), 336, 760 (App. B):
 *     Y^n_lm(th,ph) = P^n_lm(th) e^{i m ph},  P^n_lm = (-1)^n sqrt((2l+1)/4pi) d^l_{m,-n}(th),
 * zero for l < max(|m|,|n|) (eq. 40).  d is the Wigner d-function in the convention whose
 * explicit sum reproduces the App. B table (reading Q9):
 *   d^l_{m',m}(th) = sum_k (-1)^{m'-m+k} sqrt((l+m')!(l-m')!(l+m)!(l-m)!)
 *                    / ((l+m-k)! k! (m'-m+k)! (l-m'-k)!) cos^{2l+m-m'-2k}(th/2) sin^{m'-m+2k}(th/2)
 * ---------------------------------------------------------------------------------- */
static ld factl(int n) { ld f = 1; for (int q = 2; q <= n; q++) f *= q; return f; }

/* explicit sum; used (a) as the seed at l = l0 where it has a single term, (b) by the
 * tests as a second route for small l. */
static ld wigner_d_sum(int l, int mp, int m, ld th) {
    if (l < abs(mp) || l < abs(m)) return 0;
    ld c = cosl(th / 2), s = sinl(th / 2), sum = 0;
    ld pre = sqrtl(factl(l + mp) * factl(l - mp) * factl(l + m) * factl(l - m));
    for (int k = 0; k <= 2 * l; k++) {
        int a = l + m - k, b = mp - m + k, d = l - mp - k;
        if (a < 0 || b < 0 || d < 0) continue;
        ld sgn = ((mp - m + k) % 2 == 0) ? 1 : -1;
        sum += sgn * pre / (factl(a) * factl(k) * factl(b) * factl(d)) * powl(c, 2 * l + m - mp - 2 * k) * powl(s, mp - m + 2 * k);
    }
    return sum;
}
double orc_wigner_d_sum(int l, int mp, int m, double th) { return (double)wigner_d_sum(l, mp, m, (ld)th); }

/* d^l_{mp,m}(th) for l = 0..lmax by the three-term recurrence in l at fixed (mp,m), seeded at
 * l0 = max(|mp|,|m|) (where the d^{l0-1} term drops out):
 *   l sqrt(((l+1)^2-mp^2)((l+1)^2-m^2)) d^{l+1} = (2l+1)(l(l+1) x - mp m) d^l
 *                                               - (l+1) sqrt((l^2-mp^2)(l^2-m^2)) d^{l-1},  x = cos th
 * (for mp = m = 0 this is Bonnet's recurrence for Legendre polynomials, used for l0 = 0). */
static void wigner_d_rec(int lmax, int mp, int m, ld th, ld *d /* [lmax+1] */) {
    int l0 = abs(mp) > abs(m) ? abs(mp) : abs(m);
    ld x = cosl(th);
    for (int l = 0; l <= lmax; l++) d[l] = 0;
    if (l0 > lmax) return;
    d[l0] = wigner_d_sum(l0, mp, m, th);
    for (int l = l0; l < lmax; l++) {
        ld dm1 = (l > l0) ? d[l - 1] : 0;
        if (l == 0) { d[1] = x * d[0]; continue; }        /* mp = m = 0: P_1 = x P_0 */
        ld a = (ld)l * sqrtl((ld)((l + 1) * (l + 1) - mp * mp) * (ld)((l + 1) * (l + 1) - m * m));
        ld b = (ld)(2 * l + 1) * ((ld)l * (l + 1) * x - (ld)mp * m);
        ld c = (ld)(l + 1) * sqrtl((ld)(l * l - mp * mp) * (ld)(l * l - m * m));
        d[l + 1] = (b * d[l] - c * dm1) / a;
    }
}

/* P^n_lm(th) for l = 0..lmax (long double) */
static void spin_P(int n, int m, int lmax, ld th, ld *P) {
    wigner_d_rec(lmax, m, -n, th, P);
    ld sgn = (abs(n) % 2 == 0) ? 1 : -1;
    for (int l = 0; l <= lmax; l++) P[l] *= sgn * sqrtl((2 * l + 1) / (4 * PI_L));
}
void orc_spin_P(int n, int m, int lmax, double th, double *P) {
    ld *t = malloc(sizeof(ld) * (lmax + 1));
    spin_P(n, m, lmax, (ld)th, t);
    for (int l = 0; l <= lmax; l++) P[l] = (double)t[l];
    free(t);
}

/* ------------------------------------------------------------------------------------
 * Synthesis matrix (P^n_m)_{ik} = P^n_{(k+l0), m}(th_i), N x (N-l0), l0 = max(|m|,|n|)
 * (eq. 48; for n = 0, m >= 0 this is eq. 32).  The paper indexes the
 * columns from l = m; columns with l < |n| are identically zero (eq. 40) and are left out,
 * which does not change P P^+ (reading Q14).  Row-major N x ncol, long double.
 * ---------------------------------------------------------------------------------- */
static int synth_matrix(int N, int n, int m, ld *P /* N*(N-l0) */) {
    int l0 = abs(m) > abs(n) ? abs(m) : abs(n);
    int ncol = N - l0;
    if (ncol <= 0) return 0;
    ld *row = malloc(sizeof(ld) * N);
    for (int i = 0; i < N; i++) {
        spin_P(n, m, N - 1, grid_th(N, i), row);
        for (int c = 0; c < ncol; c++) P[i * ncol + c] = row[l0 + c];
    }
    free(row);
    return ncol;
}
int orc_synthesis_matrix(int N, int n, int m, double *P) {
    int l0 = abs(m) > abs(n) ? abs(m) : abs(n);
    int ncol = N - l0;
    if (ncol <= 0) return 0;
    ld *t = malloc(sizeof(ld) * N * ncol);
    synth_matrix(N, n, m, t);
    for (int p = 0; p < N * ncol; p++) P[p] = (double)t[p];
    free(t);
    return ncol;
}

/* ------------------------------------------------------------------------------------
 * O8  Filter matrix F^n_m = P f_diag P^+ (eq. 61-62; 273-285, eq. 35-36;
 * 362-366, eq. 49), reading Q11(i): analyse with the pseudo-inverse of the FULL P, zero the
 * coefficients with l > L, synthesise.  P has full column rank on these grids (Q14), so
 * P^+ s = argmin_c ||P c - s||_2, solved by Householder QR in long double.
 * F is row-major N x N, rounded once to double.  F = 0 if l0 > L.
 * ---------------------------------------------------------------------------------- */
static void filter_matrix_ld(int N, int L, int n, int m, ld *F /* N*N */) {
    int l0 = abs(m) > abs(n) ? abs(m) : abs(n);
    for (int p = 0; p < N * N; p++) F[p] = 0;
    if (l0 > L || l0 > N - 1) return;
    int nc = N - l0;
    ld *P = malloc(sizeof(ld) * N * nc), *A = malloc(sizeof(ld) * N * nc);
    ld *v = malloc(sizeof(ld) * N * nc), *beta = malloc(sizeof(ld) * nc);
    ld *b = malloc(sizeof(ld) * N), *c = malloc(sizeof(ld) * nc);
    synth_matrix(N, n, m, P);
    memcpy(A, P, sizeof(ld) * N * nc);
    /* Householder QR: A = Q R, reflectors H_q = I - beta_q v_q v_q^T stored column-wise in v */
    for (int q = 0; q < nc; q++) {
        ld nrm = 0;
        for (int i = q; i < N; i++) nrm += A[i * nc + q] * A[i * nc + q];
        nrm = sqrtl(nrm);
        ld alpha = (A[q * nc + q] > 0) ? -nrm : nrm;
        for (int i = 0; i < N; i++) v[i * nc + q] = (i < q) ? 0 : A[i * nc + q];
        v[q * nc + q] -= alpha;
        ld vv = 0;
        for (int i = q; i < N; i++) vv += v[i * nc + q] * v[i * nc + q];
        beta[q] = (vv > 0) ? 2 / vv : 0;
        for (int cc = q; cc < nc; cc++) {
            ld dot = 0;
            for (int i = q; i < N; i++) dot += v[i * nc + q] * A[i * nc + cc];
            for (int i = q; i < N; i++) A[i * nc + cc] -= beta[q] * dot * v[i * nc + q];
        }
    }
    /* column ii of F: s = e_ii;  c = R^{-1} (Q^T s)[0..nc);  zero l > L;  F[:,ii] = P c */
    for (int ii = 0; ii < N; ii++) {
        for (int i = 0; i < N; i++) b[i] = (i == ii) ? 1 : 0;
        for (int q = 0; q < nc; q++) {
            ld dot = 0;
            for (int i = q; i < N; i++) dot += v[i * nc + q] * b[i];
            for (int i = q; i < N; i++) b[i] -= beta[q] * dot * v[i * nc + q];
        }
        for (int q = nc - 1; q >= 0; q--) {
            ld s = b[q];
            for (int cc = q + 1; cc < nc; cc++) s -= A[q * nc + cc] * c[cc];
            c[q] = s / A[q * nc + q];
        }
        for (int q = 0; q < nc; q++) if (l0 + q > L) c[q] = 0;       /* f_diag, eq. 62 */
        for (int i = 0; i < N; i++) {
            ld s = 0;
            for (int q = 0; q < nc; q++) s += P[i * nc + q] * c[q];
            F[i * N + ii] = s;
        }
    }
    free(P); free(A); free(v); free(beta); free(b); free(c);
}
void orc_filter_matrix(int N, int L, int n, int m, double *F) {
    ld *t = malloc(sizeof(ld) * N * N);
    filter_matrix_ld(N, L, n, m, t);
    for (int p = 0; p < N * N; p++) F[p] = (double)t[p];
    free(t);
}
/* analysis coefficients of one theta-vector: c = P^+ s (long double QR as above), for pins */
void orc_spin_analysis(int N, int n, int m, const double *s, double *cout) {
    int l0 = abs(m) > abs(n) ? abs(m) : abs(n);
    int nc = N - l0;
    if (nc <= 0) return;
    /* build F with L = N-1 is not what is wanted here: solve directly via normal QR on [P | s] */
    ld *P = malloc(sizeof(ld) * N * nc), *A = malloc(sizeof(ld) * N * (nc + 1));
    synth_matrix(N, n, m, P);
    int w = nc + 1;
    for (int i = 0; i < N; i++) { for (int q = 0; q < nc; q++) A[i * w + q] = P[i * nc + q]; A[i * w + nc] = s[i]; }
    for (int q = 0; q < nc; q++) {
        ld nrm = 0;
        for (int i = q; i < N; i++) nrm += A[i * w + q] * A[i * w + q];
        nrm = sqrtl(nrm);
        ld alpha = (A[q * w + q] > 0) ? -nrm : nrm;
        ld *v = malloc(sizeof(ld) * N);
        for (int i = 0; i < N; i++) v[i] = (i < q) ? 0 : A[i * w + q];
        v[q] -= alpha;
        ld vv = 0;
        for (int i = q; i < N; i++) vv += v[i] * v[i];
        ld bt = (vv > 0) ? 2 / vv : 0;
        for (int cc = q; cc < w; cc++) {
            ld dot = 0;
            for (int i = q; i < N; i++) dot += v[i] * A[i * w + cc];
            for (int i = q; i < N; i++) A[i * w + cc] -= bt * dot * v[i];
        }
        free(v);
    }
    ld *c = malloc(sizeof(ld) * nc);
    for (int q = nc - 1; q >= 0; q--) {
        ld t = A[q * w + nc];
        for (int cc = q + 1; cc < nc; cc++) t -= A[q * w + cc] * c[cc];
        c[q] = t / A[q * w + q];
    }
    for (int q = 0; q < nc; q++) cout[q] = (double)c[q];
    free(P); free(A); free(c);
}

/* ------------------------------------------------------------------------------------
 * Table of filter matrices for spin weights n = -nmax..nmax and ALL m = -(N-1)..N-1, each
 * built directly from eq. (48) with that (n, m) -- no symmetry is assumed (reading Q12).
 * tab[((n+nmax)*(2N-1) + (m+N-1))*N*N + i*N + ii], double.
 * ---------------------------------------------------------------------------------- */
/* The last table is kept (it depends on (N, L, nmax) only and the time loop of O13 asks for the same
 * one thousands of times); callers must not free it. */
static double *filter_table(int N, int L, int nmax) {
    static int cN = -1, cL = -1, cn = -1;
    static double *ctab = NULL;
    if (ctab && cN == N && cL == L && cn == nmax) return ctab;
    free(ctab);
    cN = N; cL = L; cn = nmax;
    int nm = 2 * N - 1, nn = 2 * nmax + 1;
    double *tab = ctab = malloc(sizeof(double) * (size_t)nn * nm * N * N);
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int n = -nmax; n <= nmax; n++)
        for (int m = -(N - 1); m <= N - 1; m++)
            orc_filter_matrix(N, L, n, m, tab + ((size_t)(n + nmax) * nm + (m + N - 1)) * N * N);
    return tab;
}

/* ------------------------------------------------------------------------------------
 * O10  Spin-n projection filter F_n of a complex function g on ONE sphere
 * (254-259 eq. 33; 453-463 eq. 61-62; 243-246 eq. 31), complex form of
 * the real transforms (reading Q12):
 *     c_m(th_i)  = (1/J) sum_j g_ij e^{-i m ph_j},   m = -(N-1)..N-1   (m = N, Nyquist, is not
 *                                                    in the basis: PAPER.md:188-198, Q5)
 *     c~_m       = F^n_m c_m                          (real matrix on Re and Im)
 *     g~_ij      = sum_m c~_m(th_i) e^{+i m ph_j}
 * Sphere arrays are indexed [i + N*j], J = 2N.  Ftab_n points at the (2N-1) matrices of
 * this n.
 * ---------------------------------------------------------------------------------- */
static void spin_filter_sphere(int N, const double *Ftab_n, const ld *gre, const ld *gim, ld *ore, ld *oim) {
    int J = 2 * N, nm = 2 * N - 1;
    ld *cre = malloc(sizeof(ld) * nm * N), *cim = malloc(sizeof(ld) * nm * N);
    ld *dre = malloc(sizeof(ld) * nm * N), *dim_ = malloc(sizeof(ld) * nm * N);
    /* e^{i m ph_j} = e^{2 pi i q/J} with q = m j mod J: the J distinct phases, evaluated once */
    ld *cq = malloc(sizeof(ld) * J), *sq = malloc(sizeof(ld) * J);
    for (int q = 0; q < J; q++) { cq[q] = cosl(2 * PI_L * q / J); sq[q] = sinl(2 * PI_L * q / J); }
    for (int m = -(N - 1); m <= N - 1; m++)
        for (int i = 0; i < N; i++) {
            ld sr = 0, si = 0;
            for (int j = 0; j < J; j++) {
                int q = (int)((((long)m * j) % J + J) % J);
                ld c = cq[q], s = sq[q];
                sr += gre[i + N * j] * c + gim[i + N * j] * s;       /* Re g e^{-i a} */
                si += gim[i + N * j] * c - gre[i + N * j] * s;
            }
            cre[(m + N - 1) * N + i] = sr / J; cim[(m + N - 1) * N + i] = si / J;
        }
    for (int m = -(N - 1); m <= N - 1; m++) {
        const double *F = Ftab_n + (size_t)(m + N - 1) * N * N;
        for (int i = 0; i < N; i++) {
            ld sr = 0, si = 0;
            for (int ii = 0; ii < N; ii++) {
                sr += (ld)F[i * N + ii] * cre[(m + N - 1) * N + ii];
                si += (ld)F[i * N + ii] * cim[(m + N - 1) * N + ii];
            }
            dre[(m + N - 1) * N + i] = sr; dim_[(m + N - 1) * N + i] = si;
        }
    }
    for (int j = 0; j < J; j++)
        for (int i = 0; i < N; i++) {
            ld sr = 0, si = 0;
            for (int m = -(N - 1); m <= N - 1; m++) {
                int q = (int)((((long)m * j) % J + J) % J);
                ld c = cq[q], s = sq[q];
                ld a = dre[(m + N - 1) * N + i], b = dim_[(m + N - 1) * N + i];
                sr += a * c - b * s;                                  /* (a+ib) e^{+i a} */
                si += a * s + b * c;
            }
            ore[i + N * j] = sr; oim[i + N * j] = si;
        }
    free(cre); free(cim); free(dre); free(dim_); free(cq); free(sq);
}

/* public: one sphere, one spin weight, double in/out */
void orc_spin_filter_sphere(int N, int L, int n, const double *gre, const double *gim, double *ore, double *oim) {
    int J = 2 * N, nm = 2 * N - 1;
    double *tab = malloc(sizeof(double) * (size_t)nm * N * N);
#pragma omp parallel for schedule(dynamic)
    for (int m = -(N - 1); m <= N - 1; m++) orc_filter_matrix(N, L, n, m, tab + (size_t)(m + N - 1) * N * N);
    ld *a = malloc(sizeof(ld) * N * J), *b = malloc(sizeof(ld) * N * J), *c = malloc(sizeof(ld) * N * J), *d = malloc(sizeof(ld) * N * J);
    for (int p = 0; p < N * J; p++) { a[p] = gre[p]; b[p] = gim ? gim[p] : 0; }
    spin_filter_sphere(N, tab, a, b, c, d);
    for (int p = 0; p < N * J; p++) { ore[p] = (double)c[p]; oim[p] = (double)d[p]; }
    free(a); free(b); free(c); free(d); free(tab);
}

/* ------------------------------------------------------------------------------------
 * O9/O11/O12  Yn tensor filter (380-412 eq. 51-56; 422-424; 449-451 eq. 60).
 * Triad in Cartesian components (eq. 51-52):
 *     r^ = (sin th cos ph, sin th sin ph, cos th),  th^ = (cos th cos ph, cos th sin ph, -sin th),
 *     ph^ = (-sin ph, cos ph, 0),  m = (th^ + i ph^)/sqrt 2,  mbar = conj(m).
 * For every choice e = (e_1..e_k), e_q in {t (only on 4-dim indices), r^, m, mbar}:
 *     T~_e = sum_{a..} E_1[a_1] .. E_k[a_k] T^{a_1..a_k}          (eq. 56; t: E[a] = delta_{a,t})
 *     spin weight n_e = #(m) - #(mbar)                             (reading Q7, pinned by B.3)
 *     T~_e <- F_{n_e}(T~_e)                                        (O10)
 *     T'^{a..} = Re sum_e T~_e conj(E_1)[a_1] .. conj(E_k)[a_k]    (eq. 54-56; v = v_r r^ + (m.v) mbar + (mbar.v) m)
 * A t index is a spin-0 spectator (Q17).  No use is made of symmetry or conjugation: all
 * prod(dim_q) choices are filtered.
 *
 * Tensor description (flat ints): rank[t] in 0..3; dims[3t+q] in {3,4} (4: index runs t,x,y,z;
 * 3: x,y,z); sym[2t], sym[2t+1] = a symmetric index pair or -1,-1; the stored components
 * are the canonical (sym pair sorted ascending) multi-indices in row-major order, component c
 * living in field fields[foff[t] + c].
 * ksel >= 0 filters only that radius (other radii are copied through); ksel < 0: all radii.
 * ---------------------------------------------------------------------------------- */
typedef struct { ld re, im; } cld;
static cld cmul(cld a, cld b) { cld r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; return r; }

/* stored-component index of a full multi-index (row-major rank among canonical ones) */
static int comp_index(int rank, const int *dims, int s0, int s1, const int *a) {
    int idx = 0, cnt = 0, b[3], tot = 1;
    for (int q = 0; q < rank; q++) tot *= dims[q];
    int c[3] = { 0, 0, 0 };
    for (int q = 0; q < rank; q++) c[q] = a[q];
    if (s0 >= 0 && c[s0] > c[s1]) { int t = c[s0]; c[s0] = c[s1]; c[s1] = t; }
    for (int f = 0; f < tot; f++) {
        int rem = f;
        for (int q = rank - 1; q >= 0; q--) { b[q] = rem % dims[q]; rem /= dims[q]; }
        if (s0 >= 0 && b[s0] > b[s1]) continue;
        int same = 1;
        for (int q = 0; q < rank; q++) if (b[q] != c[q]) same = 0;
        if (same) { idx = cnt; break; }
        cnt++;
    }
    return idx;
}
int orc_ncomp(int rank, const int *dims, int s0, int s1) {
    int tot = 1, cnt = 0, b[3];
    for (int q = 0; q < rank; q++) tot *= dims[q];
    for (int f = 0; f < tot; f++) {
        int rem = f;
        for (int q = rank - 1; q >= 0; q--) { b[q] = rem % dims[q]; rem /= dims[q]; }
        if (s0 >= 0 && b[s0] > b[s1]) continue;
        cnt++;
    }
    return cnt;
}

static void tensor_filter_sphere(int Nr, int Nt, int Np, const double *Ftab, int nmax, int k,
                                 int rank, const int *dims, int s0, int s1, const int *fld,
                                 const double *u, double *out) {
    int N = Nt, J = Np, nm = 2 * N - 1, npt = N * J;
    int tot = 1; for (int q = 0; q < rank; q++) tot *= dims[q];
    int nchoice = 1; for (int q = 0; q < rank; q++) nchoice *= dims[q];   /* dims 4: t,r,m,mbar; 3: r,m,mbar */
    ld *accre = calloc((size_t)tot * npt, sizeof(ld));
    int *cidx = malloc(sizeof(int) * tot);               /* full multi-index -> stored component */
    for (int f = 0; f < tot; f++) {
        int a[3], r2 = f;
        for (int q = rank - 1; q >= 0; q--) { a[q] = r2 % dims[q]; r2 /= dims[q]; }
        cidx[f] = comp_index(rank, dims, s0, s1, a);
    }
    ld *gre = malloc(sizeof(ld) * npt), *gim = malloc(sizeof(ld) * npt), *fre = malloc(sizeof(ld) * npt), *fim = malloc(sizeof(ld) * npt);
    for (int e = 0; e < nchoice; e++) {
        int ch[3], rem = e, n_e = 0;                     /* ch[q]: 0 = t, 1 = r^, 2 = m, 3 = mbar */
        for (int q = rank - 1; q >= 0; q--) { ch[q] = rem % dims[q]; rem /= dims[q]; if (dims[q] == 3) ch[q] += 1; }
        for (int q = 0; q < rank; q++) { if (ch[q] == 2) n_e += 1; if (ch[q] == 3) n_e -= 1; }
        /* projection, pointwise */
        for (int j = 0; j < J; j++)
            for (int i = 0; i < N; i++) {
                ld th = grid_th(N, i), ph = grid_ph(J, j);
                ld st = sinl(th), ct = cosl(th), sp = sinl(ph), cp = cosl(ph), is2 = 1 / sqrtl(2.0L);
                cld E[4][4];                               /* E[choice][a], a = t,x,y,z */
                ld rh[4] = { 0, st * cp, st * sp, ct }, tha[4] = { 0, ct * cp, ct * sp, -st }, pha[4] = { 0, -sp, cp, 0 };
                for (int a = 0; a < 4; a++) {
                    E[0][a].re = (a == 0) ? 1 : 0; E[0][a].im = 0;
                    E[1][a].re = rh[a]; E[1][a].im = 0;
                    E[2][a].re = tha[a] * is2; E[2][a].im = pha[a] * is2;
                    E[3][a].re = tha[a] * is2; E[3][a].im = -pha[a] * is2;
                }
                cld sum = { 0, 0 };
                for (int f = 0; f < tot; f++) {
                    int a[3], r2 = f;
                    for (int q = rank - 1; q >= 0; q--) { a[q] = r2 % dims[q]; r2 /= dims[q]; }
                    cld w = { 1, 0 };
                    for (int q = 0; q < rank; q++) w = cmul(w, E[ch[q]][a[q] + (dims[q] == 3 ? 1 : 0)]);
                    ld T = u[IDX(k, i, j, fld[cidx[f]])];
                    sum.re += w.re * T; sum.im += w.im * T;
                }
                gre[i + N * j] = sum.re; gim[i + N * j] = sum.im;
            }
        spin_filter_sphere(N, Ftab + (size_t)(n_e + nmax) * nm * N * N, gre, gim, fre, fim);
        /* recombination with the conjugate dyad product, real part */
        for (int j = 0; j < J; j++)
            for (int i = 0; i < N; i++) {
                ld th = grid_th(N, i), ph = grid_ph(J, j);
                ld st = sinl(th), ct = cosl(th), sp = sinl(ph), cp = cosl(ph), is2 = 1 / sqrtl(2.0L);
                cld E[4][4];
                ld rh[4] = { 0, st * cp, st * sp, ct }, tha[4] = { 0, ct * cp, ct * sp, -st }, pha[4] = { 0, -sp, cp, 0 };
                for (int a = 0; a < 4; a++) {
                    E[0][a].re = (a == 0) ? 1 : 0; E[0][a].im = 0;
                    E[1][a].re = rh[a]; E[1][a].im = 0;
                    E[2][a].re = tha[a] * is2; E[2][a].im = -pha[a] * is2;    /* conj(m)    */
                    E[3][a].re = tha[a] * is2; E[3][a].im = pha[a] * is2;     /* conj(mbar) */
                }
                cld g = { fre[i + N * j], fim[i + N * j] };
                for (int f = 0; f < tot; f++) {
                    int a[3], r2 = f;
                    for (int q = rank - 1; q >= 0; q--) { a[q] = r2 % dims[q]; r2 /= dims[q]; }
                    cld w = g;
                    for (int q = 0; q < rank; q++) w = cmul(w, E[ch[q]][a[q] + (dims[q] == 3 ? 1 : 0)]);
                    accre[(size_t)f * npt + i + N * j] += w.re;
                }
            }
    }
    /* write every stored component once (from its canonical full multi-index) */
    for (int f = 0; f < tot; f++) {
        int a[3], r2 = f;
        for (int q = rank - 1; q >= 0; q--) { a[q] = r2 % dims[q]; r2 /= dims[q]; }
        if (s0 >= 0 && a[s0] > a[s1]) continue;
        int c = comp_index(rank, dims, s0, s1, a);
        for (int j = 0; j < J; j++)
            for (int i = 0; i < N; i++) out[IDX(k, i, j, fld[c])] = (double)accre[(size_t)f * npt + i + N * j];
    }
    free(accre); free(gre); free(gim); free(fre); free(fim); free(cidx);
}

void orc_tensor_filter(int Nr, int Nt, int Np, int L, int nfields, const double *u, double *out,
                       int ntens, const int *rank, const int *dims, const int *sym, const int *foff,
                       const int *fields, int ksel) {
    size_t tot = (size_t)Nr * Nt * Np * nfields;
    int nmax = 0;
    for (int t = 0; t < ntens; t++) {
        int ns = 0;
        for (int q = 0; q < rank[t]; q++) ns++;
        if (ns > nmax) nmax = ns;
    }
    if (out != u) memcpy(out, u, sizeof(double) * tot);
    double *Ftab = filter_table(Nt, L, nmax);
    /* one (tensor, radius) sphere per task; results are independent */
    int k0 = ksel >= 0 ? ksel : 0, k1 = ksel >= 0 ? ksel + 1 : Nr;
    double *res = (out == u) ? malloc(sizeof(double) * tot) : out;
    if (out == u) memcpy(res, u, sizeof(double) * tot);
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int t = 0; t < ntens; t++)
        for (int k = k0; k < k1; k++)
            tensor_filter_sphere(Nr, Nt, Np, Ftab, nmax, k, rank[t], dims + 3 * t, sym[2 * t], sym[2 * t + 1],
                                 fields + foff[t], u, res);
    if (out == u) { memcpy(out, res, sizeof(double) * tot); free(res); }
}

/* ------------------------------------------------------------------------------------
 * O13  First-order scalar wave system on the shell (BASELINE.json config 5).  The paper
 * has no scalar-wave system of its own; this is its class of problems, eq. (1)
 * (PAPER.md:19), specialised from the GHG first-order reduction (A.6-A.8)
 * and its characteristic machinery (A.13-A.16) to flat space
 * (readings W1-W3):
 *   u = (psi, Pi, Phi_x, Phi_y, Phi_z),  Pi = -d_t psi,  Phi_i = d_i psi
 *   d_t psi = -Pi;   d_t Pi = -(d_x Phi_x + d_y Phi_y + d_z Phi_z);   d_t Phi_i = -d_i Pi
 * Boundary shells k = 0 (outward normal s = -r^) and k = Nr-1 (s = +r^): characteristic fields
 * U^+- = Pi +- s.Phi (speeds +-1), zero-speed psi and tangential Phi.  Freeze the incoming
 * field (A.16): with d the computed RHS,  U = d_Pi + s.d_Phi;  d_Pi <- U/2;
 * d_Phi_i <- d_Phi_i - s_i (s.d_Phi) + s_i U/2;  d_psi unchanged.
 * ---------------------------------------------------------------------------------- */
void orc_wave_rhs(int Nr, int Nt, int Np, double rmin, double rmax, const double *u, double *dudt) {
    size_t npts = (size_t)Nr * Nt * Np;
    double *dg = malloc(sizeof(double) * 12 * npts);          /* [3][4]: gradient of Pi, Phi_x, Phi_y, Phi_z */
    orc_gradient(Nr, Nt, Np, 4, rmin, rmax, u + npts, dg);
    for (int j = 0; j < Np; j++)
        for (int i = 0; i < Nt; i++)
            for (int k = 0; k < Nr; k++) {
                size_t p = (size_t)k + (size_t)Nr * (i + (size_t)Nt * j);
#define DG(c, f) dg[((size_t)(c) * 4 + (f)) * npts + p]
                ld dpsi = -(ld)u[npts + p];
                ld dPi = -((ld)DG(0, 1) + (ld)DG(1, 2) + (ld)DG(2, 3));
                ld dPh[3] = { -(ld)DG(0, 0), -(ld)DG(1, 0), -(ld)DG(2, 0) };
#undef DG
                if (k == 0 || k == Nr - 1) {
                    ld th = grid_th(Nt, i), ph = grid_ph(Np, j), sg = (k == 0) ? -1 : 1;
                    ld s[3] = { sg * sinl(th) * cosl(ph), sg * sinl(th) * sinl(ph), sg * cosl(th) };
                    ld sd = s[0] * dPh[0] + s[1] * dPh[1] + s[2] * dPh[2];
                    ld U = dPi + sd;
                    dPi = U / 2;
                    for (int c = 0; c < 3; c++) dPh[c] = dPh[c] - s[c] * sd + s[c] * U / 2;
                }
                dudt[p] = (double)dpsi;
                dudt[npts + p] = (double)dPi;
                dudt[2 * npts + p] = (double)dPh[0];
                dudt[3 * npts + p] = (double)dPh[1];
                dudt[4 * npts + p] = (double)dPh[2];
            }
    free(dg);
}
