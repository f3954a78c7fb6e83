// Generalized-harmonic (GHG) right-hand side, Appendix A: (A.8)-(A.10) with gamma0 = gamma2 = 1, gamma1 = -1
// (PAPER.md:662), dependent quantities by (A.3)-(A.5) and (A.11), freezing boundary condition (A.20)-(A.21).
// Pointwise in space: one thread per grid point reads the 50 fields, their 150 Cartesian derivatives (written by
// sp_cartesian_gradient into the workspace), H_a and d_i H_a, and writes the 50 time derivatives -- 266 doubles per point,
// a few thousand flops: HBM-bound.  All index loops are over compile-time bounds and fully unrolled, symmetric pairs are
// stored once (ten components: tt,tx,ty,tz,xx,xy,xz,yy,yz,zz), the inverse metrics come from the 3+1 split
// (gamma^{ij} by cofactors, g^{tt} = -1/alpha^2, g^{ti} = beta^i/alpha^2, g^{ij} = gamma^{ij} - beta^i beta^j/alpha^2).
#pragma once
#include "sp_device.cuh"

__host__ __device__ constexpr int gsym(int a, int b) { return a <= b ? a * 4 - a * (a + 1) / 2 + b : b * 4 - b * (b + 1) / 2 + a; }
__host__ __device__ constexpr int s3(int i, int j) { return i <= j ? i * 3 - i * (i + 1) / 2 + j : j * 3 - j * (j + 1) / 2 + i; }

struct GhgArgs {
    const double *u, *du, *H, *dH;     // state [50], gradient [3][50], gauge source [4], its gradient [3][4]
    double *out;                       // d_t u [50]
    size_t npts;
};

// 3+1 split of g_ab (A.4)-(A.5): gi = gamma^{ij} (6), bu = beta^i, al = alpha, G = g^{ab} (10), nu = n^a.  false if not Lorentzian.
__device__ __forceinline__ bool ghg_split(const double (&g)[10], double (&gi)[6], double (&bu)[3], double &al, double (&G)[10],
                                          double (&nu)[4]) {
    const double gxx = g[4], gxy = g[5], gxz = g[6], gyy = g[7], gyz = g[8], gzz = g[9];
    const double cxx = gyy * gzz - gyz * gyz, cxy = gxz * gyz - gxy * gzz, cxz = gxy * gyz - gxz * gyy;
    const double cyy = gxx * gzz - gxz * gxz, cyz = gxy * gxz - gxx * gyz, czz = gxx * gyy - gxy * gxy;
    const double det = gxx * cxx + gxy * cxy + gxz * cxz;
    const double id = 1.0 / det;
    gi[0] = cxx * id; gi[1] = cxy * id; gi[2] = cxz * id; gi[3] = cyy * id; gi[4] = cyz * id; gi[5] = czz * id;
    double b2 = 0.0;
#pragma unroll
    for (int i = 0; i < 3; i++) {
        bu[i] = gi[s3(i, 0)] * g[1] + gi[s3(i, 1)] * g[2] + gi[s3(i, 2)] * g[3];
        b2 += bu[i] * g[1 + i];
    }
    const double a2 = b2 - g[0];
    al = sqrt(a2);
    const double ia2 = 1.0 / a2, ia = 1.0 / al;
    G[0] = -ia2;
    nu[0] = ia;
#pragma unroll
    for (int i = 0; i < 3; i++) {
        G[gsym(0, i + 1)] = bu[i] * ia2;
        nu[i + 1] = -bu[i] * ia;
#pragma unroll
        for (int j = i; j < 3; j++) G[gsym(i + 1, j + 1)] = gi[s3(i, j)] - bu[i] * bu[j] * ia2;
    }
    return det != 0.0 && a2 > 0.0;
}

__global__ void __launch_bounds__(128) k_ghg_rhs(GhgArgs A) {
    const size_t p = (size_t)blockIdx.x * 128 + threadIdx.x;
    if (p >= A.npts) return;
    const size_t n = A.npts;
    double g[10], k[10], d[3][10];
#pragma unroll
    for (int q = 0; q < 10; q++) {
        g[q] = A.u[(size_t)q * n + p];
        k[q] = A.u[(size_t)(10 + q) * n + p];
#pragma unroll
        for (int i = 0; i < 3; i++) d[i][q] = A.u[(size_t)(20 + 10 * i + q) * n + p];
    }
    double gi[6], bu[3], al, G[10], nu[4];
    ghg_split(g, gi, bu, al, G, nu);

    // (A.11): D[0] = d_t g_ab = -alpha k_ab + beta^i d_iab (which is (A.8) itself), D[1..3] = d_iab
    double Dt[10];
#pragma unroll
    for (int q = 0; q < 10; q++) {
        Dt[q] = -al * k[q] + bu[0] * d[0][q] + bu[1] * d[1][q] + bu[2] * d[2][q];
        A.out[(size_t)q * n + p] = Dt[q];
    }
#define GD(c, ab) ((c) == 0 ? Dt[ab] : d[(c) - 1][ab])
    // (A.3): Gamma_cab = (d_a g_bc + d_b g_ac - d_c g_ab)/2, Gamma_c = g^{ab} Gamma_cab
    double Gam[4][10], Gam1[4];
#pragma unroll
    for (int c = 0; c < 4; c++) {
        double t = 0.0;
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
            for (int b = a; b < 4; b++) {
                const double v = 0.5 * (GD(a, gsym(b, c)) + GD(b, gsym(a, c)) - GD(c, gsym(a, b)));
                Gam[c][gsym(a, b)] = v;
                t += (a == b ? 1.0 : 2.0) * G[gsym(a, b)] * v;
            }
        Gam1[c] = t;
    }
#undef GD
    double Hh[4], Hup[4], Cc[4], nC = 0.0;
#pragma unroll
    for (int a = 0; a < 4; a++) Hh[a] = A.H[(size_t)a * n + p];
#pragma unroll
    for (int a = 0; a < 4; a++) {
        Hup[a] = G[gsym(a, 0)] * Hh[0] + G[gsym(a, 1)] * Hh[1] + G[gsym(a, 2)] * Hh[2] + G[gsym(a, 3)] * Hh[3];
        Cc[a] = Hh[a] + Gam1[a];                       // H_c + Gamma_c
        nC += nu[a] * Cc[a];
    }
    // scalars and small vectors of the source terms
    double nnk = 0.0, nk[3] = {0.0, 0.0, 0.0}, nkd[3], nnd[3], M[3][3];
#pragma unroll
    for (int c = 0; c < 4; c++)
#pragma unroll
        for (int e = 0; e < 4; e++) nnk += nu[c] * nu[e] * k[gsym(c, e)];
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int c = 0; c < 4; c++) nk[i] += nu[c] * k[gsym(c, i + 1)];          // n^c k_ci
#pragma unroll
    for (int j = 0; j < 3; j++) nkd[j] = gi[s3(0, j)] * nk[0] + gi[s3(1, j)] * nk[1] + gi[s3(2, j)] * nk[2];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        double t = 0.0, nd[3] = {0.0, 0.0, 0.0};
#pragma unroll
        for (int c = 0; c < 4; c++) {
#pragma unroll
            for (int e = 0; e < 4; e++) t += nu[c] * nu[e] * d[i][gsym(c, e)];
#pragma unroll
            for (int j = 0; j < 3; j++) nd[j] += nu[c] * d[i][gsym(j + 1, c)];   // n^c d_ijc
        }
        nnd[i] = t;
#pragma unroll
        for (int kk = 0; kk < 3; kk++) M[i][kk] = gi[s3(0, kk)] * nd[0] + gi[s3(1, kk)] * nd[1] + gi[s3(2, kk)] * nd[2];
    }
    // quadratic terms of (A.10): Q_ab = g^{cd} (gamma^{ij} d_iac d_jbd - k_ac k_bd - g^{ef} Gamma_ace Gamma_bdf)
    double Q[10];
#pragma unroll
    for (int q = 0; q < 10; q++) Q[q] = 0.0;
#pragma unroll
    for (int a = 0; a < 4; a++) {
        double U[10], F[3][4], Kd[4];
        {   // U_a^{df} = g^{cd} g^{ef} Gamma_{a,ce}
            double V[4][4];
#pragma unroll
            for (int dd = 0; dd < 4; dd++)
#pragma unroll
                for (int e = 0; e < 4; e++)
                    V[dd][e] = G[gsym(0, dd)] * Gam[a][gsym(0, e)] + G[gsym(1, dd)] * Gam[a][gsym(1, e)] +
                               G[gsym(2, dd)] * Gam[a][gsym(2, e)] + G[gsym(3, dd)] * Gam[a][gsym(3, e)];
#pragma unroll
            for (int dd = 0; dd < 4; dd++)
#pragma unroll
                for (int f = dd; f < 4; f++)
                    U[gsym(dd, f)] = G[gsym(0, f)] * V[dd][0] + G[gsym(1, f)] * V[dd][1] + G[gsym(2, f)] * V[dd][2] + G[gsym(3, f)] * V[dd][3];
        }
        {   // F^j_a^d = gamma^{ij} g^{cd} d_iac
            double E[3][4];
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int dd = 0; dd < 4; dd++)
                    E[i][dd] = G[gsym(0, dd)] * d[i][gsym(a, 0)] + G[gsym(1, dd)] * d[i][gsym(a, 1)] + G[gsym(2, dd)] * d[i][gsym(a, 2)] +
                               G[gsym(3, dd)] * d[i][gsym(a, 3)];
#pragma unroll
            for (int j = 0; j < 3; j++)
#pragma unroll
                for (int dd = 0; dd < 4; dd++) F[j][dd] = gi[s3(0, j)] * E[0][dd] + gi[s3(1, j)] * E[1][dd] + gi[s3(2, j)] * E[2][dd];
        }
#pragma unroll
        for (int dd = 0; dd < 4; dd++)
            Kd[dd] = G[gsym(0, dd)] * k[gsym(a, 0)] + G[gsym(1, dd)] * k[gsym(a, 1)] + G[gsym(2, dd)] * k[gsym(a, 2)] + G[gsym(3, dd)] * k[gsym(a, 3)];
#pragma unroll
        for (int b = a; b < 4; b++) {
            double t = 0.0;
#pragma unroll
            for (int dd = 0; dd < 4; dd++) {
#pragma unroll
                for (int j = 0; j < 3; j++) t += F[j][dd] * d[j][gsym(b, dd)];
                t -= Kd[dd] * k[gsym(b, dd)];
#pragma unroll
                for (int f = 0; f < 4; f++) t -= U[gsym(dd, f)] * Gam[b][gsym(dd, f)];
            }
            Q[gsym(a, b)] = t;
        }
    }
    // per component: algebraic source terms plus the derivative terms of (A.9), (A.10)
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
        for (int b = a; b < 4; b++) {
            const int q = gsym(a, b);
            // 2 nabla_(a H_b) = d_a H_b + d_b H_a - 2 g^{cd} Gamma_cab H_d, with d_t H = 0 (A.18)
            double nab = -2.0 * (Hup[0] * Gam[0][q] + Hup[1] * Gam[1][q] + Hup[2] * Gam[2][q] + Hup[3] * Gam[3][q]);
            if (a > 0) nab += A.dH[(size_t)((a - 1) * 4 + b) * n + p];
            if (b > 0) nab += A.dH[(size_t)((b - 1) * 4 + a) * n + p];
            const double nb = (b == 0) ? -al : 0.0, na = (a == 0) ? -al : 0.0;     // n_a = (-alpha, 0, 0, 0)
            double tk = 2.0 * al * Q[q] - al * nab - 0.5 * al * nnk * k[q] - al * (nkd[0] * d[0][q] + nkd[1] * d[1][q] + nkd[2] * d[2][q]) +
                        al * (nb * Cc[a] + na * Cc[b] - g[q] * nC) + (bu[0] * d[0][q] + bu[1] * d[1][q] + bu[2] * d[2][q]);
            double td[3];
#pragma unroll
            for (int i = 0; i < 3; i++)
                td[i] = 0.5 * al * nnd[i] * k[q] + al * (M[i][0] * d[0][q] + M[i][1] * d[1][q] + M[i][2] * d[2][q]) - al * d[i][q];
#pragma unroll
            for (int kk = 0; kk < 3; kk++) {
                const double dgk = A.du[(size_t)(kk * 50 + q) * n + p], dkk = A.du[(size_t)(kk * 50 + 10 + q) * n + p];
                double ddk[3];
#pragma unroll
                for (int i = 0; i < 3; i++) ddk[i] = A.du[(size_t)(kk * 50 + 20 + 10 * i + q) * n + p];
                tk += bu[kk] * (dkk - dgk) - al * (gi[s3(0, kk)] * ddk[0] + gi[s3(1, kk)] * ddk[1] + gi[s3(2, kk)] * ddk[2]);
#pragma unroll
                for (int i = 0; i < 3; i++) td[i] += bu[kk] * ddk[i];
                td[kk] += al * (dgk - dkk);
            }
            A.out[(size_t)(10 + q) * n + p] = tk;
#pragma unroll
            for (int i = 0; i < 3; i++) A.out[(size_t)(20 + 10 * i + q) * n + p] = td[i];
        }
}

// Freezing boundary condition (A.20)-(A.21) on the outer shell k = Nr-1: one thread per (i, j).
// s_i = l_i / sqrt(gamma^{ij} l_i l_j), l = x_i / r, s^k = gamma^{kj} s_j.
__global__ void k_ghg_bc(const double *__restrict__ u, double *__restrict__ out, size_t npts, int Nr, int Nt, int Np,
                         const double *__restrict__ sin_t, const double *__restrict__ cos_t, const double *__restrict__ sin_p,
                         const double *__restrict__ cos_p) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= Nt * Np) return;
    const int i = q % Nt, j = q / Nt;
    const size_t p = (size_t)(Nr - 1) + (size_t)Nr * (i + (size_t)Nt * j);
    double g[10], gi[6], bu[3], al, G[10], nu[4];
#pragma unroll
    for (int c = 0; c < 10; c++) g[c] = u[(size_t)c * npts + p];
    ghg_split(g, gi, bu, al, G, nu);
    const double l[3] = {sin_t[i] * cos_p[j], sin_t[i] * sin_p[j], cos_t[i]};
    double nrm = 0.0;
#pragma unroll
    for (int x = 0; x < 3; x++)
#pragma unroll
        for (int y = 0; y < 3; y++) nrm += gi[s3(x, y)] * l[x] * l[y];
    nrm = sqrt(nrm);
    double sd[3], su[3];
#pragma unroll
    for (int x = 0; x < 3; x++) sd[x] = l[x] / nrm;
#pragma unroll
    for (int x = 0; x < 3; x++) su[x] = gi[s3(x, 0)] * sd[0] + gi[s3(x, 1)] * sd[1] + gi[s3(x, 2)] * sd[2];
    for (int c = 0; c < 10; c++) {
        const double g0 = out[(size_t)c * npts + p], k0 = out[(size_t)(10 + c) * npts + p];
        const double s = su[0] * out[(size_t)(20 + c) * npts + p] + su[1] * out[(size_t)(30 + c) * npts + p] + su[2] * out[(size_t)(40 + c) * npts + p];
        out[(size_t)(10 + c) * npts + p] = 0.5 * (g0 + k0 + s);
        const double w = 0.5 * (-g0 + k0 + s);
#pragma unroll
        for (int x = 0; x < 3; x++) out[(size_t)(20 + 10 * x + c) * npts + p] = sd[x] * w;
    }
}

// Initial data from a metric with d_t g_ab = 0: k_ab = (beta^i/alpha) d_iab by (A.6), H_a = -Gamma_a (A.18).
__global__ void __launch_bounds__(128) k_ghg_init(double *u, double *H, size_t npts) {
    const size_t p = (size_t)blockIdx.x * 128 + threadIdx.x;
    if (p >= npts) return;
    const size_t n = npts;
    double g[10], k[10], d[3][10], gi[6], bu[3], al, G[10], nu[4], Dt[10];
#pragma unroll
    for (int q = 0; q < 10; q++) {
        g[q] = u[(size_t)q * n + p];
#pragma unroll
        for (int i = 0; i < 3; i++) d[i][q] = u[(size_t)(20 + 10 * i + q) * n + p];
    }
    ghg_split(g, gi, bu, al, G, nu);
#pragma unroll
    for (int q = 0; q < 10; q++) {
        k[q] = (bu[0] * d[0][q] + bu[1] * d[1][q] + bu[2] * d[2][q]) / al;
        u[(size_t)(10 + q) * n + p] = k[q];
        Dt[q] = -al * k[q] + bu[0] * d[0][q] + bu[1] * d[1][q] + bu[2] * d[2][q];
    }
#define GD(c, ab) ((c) == 0 ? Dt[ab] : d[(c) - 1][ab])
#pragma unroll
    for (int c = 0; c < 4; c++) {
        double t = 0.0;
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
            for (int b = a; b < 4; b++)
                t += (a == b ? 1.0 : 2.0) * G[gsym(a, b)] * 0.5 * (GD(a, gsym(b, c)) + GD(b, gsym(a, c)) - GD(c, gsym(a, b)));
        H[(size_t)c * n + p] = -t;
    }
#undef GD
}
