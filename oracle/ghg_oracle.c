/* CPU oracle for the generalized-harmonic (GHG) right-hand side of PAPER.md Appendix A
 * (SURVEY.md 8(f) NEXT-1).  TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline leg may call it; it shares no code with the CUDA library.
 *
 * Plain index notation, every sum written as a loop over the indices the paper prints, long
 * double arithmetic, full 4x4 / 3x3 arrays (no use of the symmetry to save work), inverse
 * metrics by Gauss-Jordan elimination "from the component matrices".
 *
 * State layout: 50 fields, each state-shaped [Np][Nt][Nr]:
 *     g_ab   fields  0.. 9   (ab = tt,tx,ty,tz,xx,xy,xz,yy,yz,zz)
 *     k_ab   fields 10..19   (the paper's k_ab = -n^c d_c g_ab, eq. A.6; "Pi_ab" of the survey)
 *     d_iab  fields 20..49   (i = x,y,z slowest, then the same ten)
 * du = Cartesian gradient of the state, [3][50] state-shaped (du[c][mu] = d_c u^mu, c = x,y,z);
 * H = gauge source H_a, [4]; dH = its spatial gradient [3][4] (d_t H_a = 0, eq. A.18).
 *
 * What is implemented, as printed:
 *   orc_ghg_rhs      (A.8), (A.9), (A.10) with gamma0 = gamma2 = 1, gamma1 = -1,
 *                    dependent quantities by (A.3)-(A.5), (A.11), nabla_a H_b of PAPER.md:682;
 *                    optionally the freezing boundary condition (A.20)-(A.21) on the shell
 *                    k = Nr-1, with s_i the outward normal x_i/r normalised by gamma^{ij}
 *                    (PAPER.md:746).
 *   orc_ghg_init     k_ab from (A.6) with d_t g_ab = 0 and H_a = -Gamma_a from (A.18), (A.3).
 * Pins (tests/test_oracle_ghg.py): the Kerr-Schild metric (A.17) is a static solution of the
 * Einstein equations, so the RHS of data built from it -- for the centred hole and for a hole
 * displaced from the origin, which breaks every symmetry of the grid -- must vanish to the
 * truncation error of the spectral derivatives and fall exponentially with Nr (a dropped term,
 * wrong sign or misplaced index in any term that does NOT vanish on constraint-satisfying data
 * leaves an O(1) residual that does not converge); Minkowski gives exactly zero; alpha, beta^i,
 * gamma^{ij} against the closed forms (A.19); with the boundary condition on, the incoming
 * characteristic combinations of (A.14) vanish and the outgoing one and d_t g_ab are those of
 * the unconstrained RHS.  The terms proportional to the constraints d_i g_ab - d_iab and
 * H_a + Gamma_a (+alpha d_i g_ab, -alpha d_iab in (A.9); -beta^k d_k g_ab, +beta^i d_iab and the
 * gamma0 term in (A.10)) are silent on that data; they are pinned one by one through the closed-form
 * linear response on a flat background (Minkowski and Minkowski in shifted coordinates), each
 * test checked to fail when the sign of its term is flipped.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef long double ld;
#define PI_L 3.141592653589793238462643383279502884L

static const int SYM[4][4] = {{0, 1, 2, 3}, {1, 4, 5, 6}, {2, 5, 7, 8}, {3, 6, 8, 9}};

static int inv_gauss_jordan(int n, const ld *A, ld *Ai) {
    ld M[4][8];
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) { M[i][j] = A[i * n + j]; M[i][n + j] = (i == j) ? 1.0L : 0.0L; }
    for (int c = 0; c < n; c++) {
        int piv = c;
        for (int r = c + 1; r < n; r++) if (fabsl(M[r][c]) > fabsl(M[piv][c])) piv = r;
        if (M[piv][c] == 0.0L) return 1;
        if (piv != c) for (int j = 0; j < 2 * n; j++) { ld t = M[c][j]; M[c][j] = M[piv][j]; M[piv][j] = t; }
        ld d = M[c][c];
        for (int j = 0; j < 2 * n; j++) M[c][j] /= d;
        for (int r = 0; r < n; r++) if (r != c) {
            ld f = M[r][c];
            for (int j = 0; j < 2 * n; j++) M[r][j] -= f * M[c][j];
        }
    }
    for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) Ai[i * n + j] = M[i][n + j];
    return 0;
}

/* everything the equations need at one point */
typedef struct {
    ld g[4][4], k[4][4], d[3][4][4];          /* d[i][a][b] = d_iab                                  */
    ld ginv[4][4], gam_inv[3][3];             /* g^{ab}, gamma^{ij}                                  */
    ld alpha, beta_up[3], n_up[4], n_dn[4];   /* (A.4), (A.5)                                        */
    ld D[4][4][4];                            /* D[c][a][b] = d_c g_ab by (A.11), c = t,x,y,z        */
    ld Gam[4][4][4];                          /* Gam[c][a][b] = Gamma_cab (A.3)                      */
    ld Gam1[4];                               /* Gamma_c = g^{ab} Gamma_cab                          */
} ghg_point;

static int ghg_dependent(ghg_point *q) {
    ld gam[9], gi[9], g4[16], g4i[16];
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) gam[i * 3 + j] = q->g[i + 1][j + 1];   /* gamma_ij = g_ij */
    if (inv_gauss_jordan(3, gam, gi)) return 1;
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) q->gam_inv[i][j] = gi[i * 3 + j];
    for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) g4[a * 4 + b] = q->g[a][b];
    if (inv_gauss_jordan(4, g4, g4i)) return 1;
    for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) q->ginv[a][b] = g4i[a * 4 + b];
    ld b2 = 0;
    for (int i = 0; i < 3; i++) {                      /* beta_i = g_ti, beta^i = gamma^{ij} beta_j */
        q->beta_up[i] = 0;
        for (int j = 0; j < 3; j++) q->beta_up[i] += q->gam_inv[i][j] * q->g[0][j + 1];
    }
    for (int i = 0; i < 3; i++) b2 += q->g[0][i + 1] * q->beta_up[i];
    ld a2 = b2 - q->g[0][0];                           /* alpha = sqrt(beta_i beta^i - g_tt) */
    if (!(a2 > 0)) return 1;
    q->alpha = sqrtl(a2);
    q->n_dn[0] = -q->alpha; q->n_dn[1] = q->n_dn[2] = q->n_dn[3] = 0;        /* (A.4) */
    q->n_up[0] = 1 / q->alpha;
    for (int i = 0; i < 3; i++) q->n_up[i + 1] = -q->beta_up[i] / q->alpha;
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {                  /* (A.11) */
            ld t = -q->alpha * q->k[a][b];
            for (int i = 0; i < 3; i++) t += q->beta_up[i] * q->d[i][a][b];
            q->D[0][a][b] = t;
            for (int i = 0; i < 3; i++) q->D[i + 1][a][b] = q->d[i][a][b];
        }
    for (int c = 0; c < 4; c++)                        /* (A.3) */
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++) q->Gam[c][a][b] = 0.5L * (q->D[a][b][c] + q->D[b][a][c] - q->D[c][a][b]);
    for (int c = 0; c < 4; c++) {
        ld t = 0;
        for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) t += q->ginv[a][b] * q->Gam[c][a][b];
        q->Gam1[c] = t;
    }
    return 0;
}

static void load_point(const double *u, size_t npts, size_t p, ghg_point *q) {
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {
            q->g[a][b] = u[(size_t)SYM[a][b] * npts + p];
            q->k[a][b] = u[(size_t)(10 + SYM[a][b]) * npts + p];
            for (int i = 0; i < 3; i++) q->d[i][a][b] = u[(size_t)(20 + 10 * i + SYM[a][b]) * npts + p];
        }
}

/* (A.8)-(A.10) at one point.  dg[k][a][b] = d_k g_ab, dk[k][a][b] = d_k k_ab, dd[k][i][a][b] = d_k d_iab (numerical
 * derivatives of the state), H[a], dH[k][a] = d_k H_a.  Outputs tg, tk, td = d_t of g, k, d. */
static void ghg_rhs_point(const ghg_point *q, ld dg[3][4][4], ld dk[3][4][4], ld dd[3][3][4][4], const ld H[4], ld dH[3][4],
                          ld tg[4][4], ld tk[4][4], ld td[3][4][4]) {
    const ld al = q->alpha;
    /* nabla_a H_b = d_a H_b - g^{cd} Gamma_cab H_d, d_t H_b = 0 (A.18) */
    ld nabH[4][4];
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {
            ld t = (a == 0) ? 0.0L : dH[a - 1][b];
            for (int c = 0; c < 4; c++) for (int e = 0; e < 4; e++) t -= q->ginv[c][e] * q->Gam[c][a][b] * H[e];
            nabH[a][b] = t;
        }
    ld C[4];                                           /* H_c + Gamma_c */
    for (int c = 0; c < 4; c++) C[c] = H[c] + q->Gam1[c];
    ld nnk = 0;                                        /* n^c n^d k_cd */
    for (int c = 0; c < 4; c++) for (int e = 0; e < 4; e++) nnk += q->n_up[c] * q->n_up[e] * q->k[c][e];
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {
            /* (A.8) */
            ld t8 = -al * q->k[a][b];
            for (int i = 0; i < 3; i++) t8 += q->beta_up[i] * q->d[i][a][b];
            tg[a][b] = t8;
            /* (A.9) */
            for (int i = 0; i < 3; i++) {
                ld t = 0;
                for (int kk = 0; kk < 3; kk++) t += q->beta_up[kk] * dd[kk][i][a][b];
                t += -al * dk[i][a][b] + al * dg[i][a][b];
                ld nnd = 0;                            /* n^c n^d d_icd */
                for (int c = 0; c < 4; c++) for (int e = 0; e < 4; e++) nnd += q->n_up[c] * q->n_up[e] * q->d[i][c][e];
                t += 0.5L * al * nnd * q->k[a][b];
                for (int j = 0; j < 3; j++)
                    for (int kk = 0; kk < 3; kk++) {
                        ld nd = 0;                     /* n^c d_ijc */
                        for (int c = 0; c < 4; c++) nd += q->n_up[c] * q->d[i][j + 1][c];
                        t += al * q->gam_inv[j][kk] * nd * q->d[kk][a][b];
                    }
                t -= al * q->d[i][a][b];
                td[i][a][b] = t;
            }
            /* (A.10) */
            ld t = 0;
            for (int kk = 0; kk < 3; kk++) t += q->beta_up[kk] * dk[kk][a][b];
            for (int i = 0; i < 3; i++) for (int kk = 0; kk < 3; kk++) t -= al * q->gam_inv[i][kk] * dd[kk][i][a][b];
            for (int kk = 0; kk < 3; kk++) t -= q->beta_up[kk] * dg[kk][a][b];
            for (int c = 0; c < 4; c++)
                for (int e = 0; e < 4; e++) {
                    ld in = 0;
                    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) in += q->gam_inv[i][j] * q->d[i][a][c] * q->d[j][b][e];
                    in -= q->k[a][c] * q->k[b][e];
                    for (int x = 0; x < 4; x++) for (int y = 0; y < 4; y++) in -= q->ginv[x][y] * q->Gam[a][c][x] * q->Gam[b][e][y];
                    t += 2 * al * q->ginv[c][e] * in;
                }
            t -= al * (nabH[a][b] + nabH[b][a]);       /* 2 alpha nabla_(a H_b) */
            t -= 0.5L * al * nnk * q->k[a][b];
            for (int c = 0; c < 4; c++)
                for (int i = 0; i < 3; i++)
                    for (int j = 0; j < 3; j++) t -= al * q->n_up[c] * q->k[c][i + 1] * q->gam_inv[i][j] * q->d[j][a][b];
            {
                ld nC = 0;
                for (int c = 0; c < 4; c++) nC += q->n_up[c] * C[c];
                t += al * (q->n_dn[b] * C[a] + q->n_dn[a] * C[b] - q->g[a][b] * nC);   /* 2 delta^c_(a n_b) - g_ab n^c */
            }
            for (int i = 0; i < 3; i++) t += q->beta_up[i] * q->d[i][a][b];
            tk[a][b] = t;
        }
}

/* u [50], du [3][50], H [4], dH [3][4] -> dudt [50].  bc_outer != 0: (A.20)-(A.21) on k = Nr-1.
 * Returns the number of points where the metric is not invertible / alpha^2 <= 0 (0 = fine). */
int orc_ghg_rhs(int Nr, int Nt, int Np, double rmin, double rmax, const double *u, const double *du, const double *H,
                const double *dH, int bc_outer, double *dudt) {
    const size_t npts = (size_t)Nr * Nt * Np;
    int bad = 0;
    (void)rmin; (void)rmax;
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (long pp = 0; pp < (long)npts; pp++) {
        const size_t p = (size_t)pp;
        ghg_point q;
        load_point(u, npts, p, &q);
        if (ghg_dependent(&q)) { bad++; for (int f = 0; f < 50; f++) dudt[(size_t)f * npts + p] = 0; continue; }
        ld dg[3][4][4], dk[3][4][4], dd[3][3][4][4], Hh[4], dHh[3][4], tg[4][4], tk[4][4], td[3][4][4];
        for (int c = 0; c < 3; c++)
            for (int a = 0; a < 4; a++) {
                dHh[c][a] = dH[((size_t)c * 4 + a) * npts + p];
                for (int b = 0; b < 4; b++) {
                    dg[c][a][b] = du[((size_t)c * 50 + SYM[a][b]) * npts + p];
                    dk[c][a][b] = du[((size_t)c * 50 + 10 + SYM[a][b]) * npts + p];
                    for (int i = 0; i < 3; i++) dd[c][i][a][b] = du[((size_t)c * 50 + 20 + 10 * i + SYM[a][b]) * npts + p];
                }
            }
        for (int a = 0; a < 4; a++) Hh[a] = H[(size_t)a * npts + p];
        ghg_rhs_point(&q, dg, dk, dd, Hh, dHh, tg, tk, td);
        const int kr = (int)(p % (size_t)Nr);
        if (bc_outer && kr == Nr - 1) {
            /* outward normal: s_i = l_i / sqrt(gamma^{ij} l_i l_j), l_i = x_i / r;  s^k = gamma^{kj} s_j */
            const int i = (int)((p / (size_t)Nr) % (size_t)Nt), j = (int)(p / ((size_t)Nr * Nt));
            const ld th = PI_L * (i + 0.5L) / Nt, ph = 2 * PI_L * j / Np;
            ld l[3] = {sinl(th) * cosl(ph), sinl(th) * sinl(ph), cosl(th)}, s_dn[3], s_up[3], nrm = 0;
            for (int x = 0; x < 3; x++) for (int y = 0; y < 3; y++) nrm += q.gam_inv[x][y] * l[x] * l[y];
            nrm = sqrtl(nrm);
            for (int x = 0; x < 3; x++) s_dn[x] = l[x] / nrm;
            for (int x = 0; x < 3; x++) { s_up[x] = 0; for (int y = 0; y < 3; y++) s_up[x] += q.gam_inv[x][y] * s_dn[y]; }
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++) {
                    ld sd = 0;
                    for (int x = 0; x < 3; x++) sd += s_up[x] * td[x][a][b];
                    const ld g0 = tg[a][b], k0 = tk[a][b];
                    tk[a][b] = 0.5L * (g0 + k0 + sd);                                  /* (A.20) */
                    for (int x = 0; x < 3; x++) td[x][a][b] = 0.5L * s_dn[x] * (-g0 + k0 + sd);   /* (A.21) */
                }
        }
        for (int a = 0; a < 4; a++)
            for (int b = a; b < 4; b++) {
                dudt[(size_t)SYM[a][b] * npts + p] = (double)tg[a][b];
                dudt[(size_t)(10 + SYM[a][b]) * npts + p] = (double)tk[a][b];
                for (int i = 0; i < 3; i++) dudt[(size_t)(20 + 10 * i + SYM[a][b]) * npts + p] = (double)td[i][a][b];
            }
    }
    return bad;
}

/* Initial data from a metric with d_t g_ab = 0: on entry u holds g_ab (fields 0..9) and
 * d_iab (fields 20..49, e.g. the numerical gradient of g_ab); fills k_ab = (beta^i / alpha) d_iab  ((A.6) with
 * d_t g_ab = 0) and H_a = -Gamma_a (A.18).  Returns the number of bad points. */
int orc_ghg_init(int Nr, int Nt, int Np, double *u, double *H) {
    const size_t npts = (size_t)Nr * Nt * Np;
    int bad = 0;
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (long pp = 0; pp < (long)npts; pp++) {
        const size_t p = (size_t)pp;
        ghg_point q;
        load_point(u, npts, p, &q);
        for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) q.k[a][b] = 0;
        if (ghg_dependent(&q)) { bad++; continue; }
        for (int a = 0; a < 4; a++)
            for (int b = a; b < 4; b++) {
                ld t = 0;
                for (int i = 0; i < 3; i++) t += q.beta_up[i] * q.d[i][a][b];
                q.k[a][b] = q.k[b][a] = t / q.alpha;
                u[(size_t)(10 + SYM[a][b]) * npts + p] = (double)(t / q.alpha);
            }
        /* with this k, (A.11) gives d_t g = 0; recompute Gamma_a with it */
        for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) q.k[a][b] = u[(size_t)(10 + SYM[a][b]) * npts + p];
        ghg_dependent(&q);
        for (int a = 0; a < 4; a++) H[(size_t)a * npts + p] = (double)(-q.Gam1[a]);
    }
    return bad;
}

/* 3+1 quantities of (A.4)-(A.5) at every point, for the closed-form pin (A.19): out = [alpha, beta^x, beta^y, beta^z,
 * gamma^{xx}, gamma^{xy}, gamma^{xz}, gamma^{yy}, gamma^{yz}, gamma^{zz}] state-shaped. */
int orc_ghg_lapse_shift(int Nr, int Nt, int Np, const double *u, double *out) {
    const size_t npts = (size_t)Nr * Nt * Np;
    int bad = 0;
    for (size_t p = 0; p < npts; p++) {
        ghg_point q;
        load_point(u, npts, p, &q);
        if (ghg_dependent(&q)) { bad++; continue; }
        out[p] = (double)q.alpha;
        for (int i = 0; i < 3; i++) out[(size_t)(1 + i) * npts + p] = (double)q.beta_up[i];
        int c = 4;
        for (int i = 0; i < 3; i++) for (int j = i; j < 3; j++) out[(size_t)(c++) * npts + p] = (double)q.gam_inv[i][j];
    }
    return bad;
}
