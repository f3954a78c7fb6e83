// First-order scalar wave system on the shell (BASELINE.json config 5; readings W1-W3).
//   u = (psi, Pi, Phi_x, Phi_y, Phi_z):  d_t psi = -Pi;  d_t Pi = -d_i Phi_i;  d_t Phi_i = -d_i Pi
// (psi <-> g, Pi <-> k, Phi_i <-> d_i in PAPER.md:666-670, 700 (A.7, A.8, A.13) with flat background).
// Boundary shells k = 0 (s = -r^) and k = Nr-1 (s = +r^): freeze the incoming characteristic field
// U^- = Pi - s.Phi, keep U^+ = Pi + s.Phi and the zero-speed fields (A.16):
//   d_Pi <- (d_Pi + s.d_Phi)/2,   d_Phi_i <- d_Phi_i + s_i (d_Pi - s.d_Phi)/2.
#pragma once
#include "sp_device.cuh"

// dg: gradient of the 4 fields (Pi, Phi_x, Phi_y, Phi_z), [3][4] state-shaped
__global__ void __launch_bounds__(256)
k_wave_rhs(int Nr, int Nt, size_t npts, const double *__restrict__ sin_t, const double *__restrict__ cos_t,
           const double *__restrict__ sin_p, const double *__restrict__ cos_p, const double *__restrict__ u,
           const double *__restrict__ dg, double *__restrict__ dudt, int bcmask) {
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npts) return;
    const int k = (int)(p % Nr), i = (int)((p / Nr) % Nt), j = (int)(p / ((size_t)Nr * Nt));
    auto D = [&](int c, int f) { return dg[((size_t)c * 4 + f) * npts + p]; };
    double dpsi = -u[npts + p];
    double dPi = -(D(0, 1) + D(1, 2) + D(2, 3));
    double dPh[3] = {-D(0, 0), -D(1, 0), -D(2, 0)};
    if ((k == 0 && (bcmask & 1)) || (k == Nr - 1 && (bcmask & 2))) {      // bcmask: bit 0 inner, bit 1 outer sphere is a physical boundary
        const double sg = (k == 0) ? -1.0 : 1.0;
        const double s[3] = {sg * sin_t[i] * cos_p[j], sg * sin_t[i] * sin_p[j], sg * cos_t[i]};
        const double sd = s[0] * dPh[0] + s[1] * dPh[1] + s[2] * dPh[2];
        const double h = 0.5 * (dPi - sd);
        dPi = 0.5 * (dPi + sd);
#pragma unroll
        for (int c = 0; c < 3; c++) dPh[c] += s[c] * h;
    }
    dudt[p] = dpsi;
    dudt[npts + p] = dPi;
    dudt[2 * npts + p] = dPh[0];
    dudt[3 * npts + p] = dPh[1];
    dudt[4 * npts + p] = dPh[2];
}

// Characteristic coupling of two shells on their shared sphere (spshell.h: sp_wave_interface).  One thread per (i, j); a = the inner
// shell's RHS row k = Nra-1, b = the outer shell's row k = 0, both raw on entry.
__global__ void __launch_bounds__(128)
k_wave_interface(int Nt, int Np, int Nra, int Nrb, const double *__restrict__ sin_t, const double *__restrict__ cos_t,
                 const double *__restrict__ sin_p, const double *__restrict__ cos_p, double *da, double *db) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= Nt * Np) return;
    const int i = q % Nt, j = q / Nt;
    const size_t na = (size_t)Nra * Nt * Np, nb = (size_t)Nrb * Nt * Np;
    const size_t pa = (size_t)q * Nra + (Nra - 1), pb = (size_t)q * Nrb;
    const double n[3] = {sin_t[i] * cos_p[j], sin_t[i] * sin_p[j], cos_t[i]};
    const double aPi = da[na + pa], bPi = db[nb + pb];
    double aPh[3], bPh[3];
#pragma unroll
    for (int c = 0; c < 3; c++) { aPh[c] = da[(2 + c) * na + pa]; bPh[c] = db[(2 + c) * nb + pb]; }
    const double nA = n[0] * aPh[0] + n[1] * aPh[1] + n[2] * aPh[2], nB = n[0] * bPh[0] + n[1] * bPh[1] + n[2] * bPh[2];
    const double Up = aPi + nA, Um = bPi - nB;          // leaves the inner shell outward / leaves the outer shell inward
    const double dPi = 0.5 * (Up + Um), nd = 0.5 * (Up - Um);
    da[na + pa] = dPi; db[nb + pb] = dPi;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        da[(2 + c) * na + pa] = aPh[c] + n[c] * (nd - nA);
        db[(2 + c) * nb + pb] = bPh[c] + n[c] * (nd - nB);
    }
}

__global__ void __launch_bounds__(256) k_axpby(double a, const double *__restrict__ x, double b, double *__restrict__ y, size_t n) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += stride) y[q] = a * x[q] + b * y[q];
}

// One RK4 combination: acc_out = acc_in + c_acc * k  and, if stage_out is given, stage_out = u + c_stage * k.
// u and k are read once; acc_out may alias acc_in or u (same index read before written by the same thread).
__global__ void __launch_bounds__(256) k_rk4_stage(const double *u, const double *__restrict__ k, const double *acc_in,
                                                   double *acc_out, double *stage_out, double c_acc, double c_stage, size_t n) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += stride) {
        const double kq = k[q], uq = u[q];
        const double a = (acc_in == u) ? uq : acc_in[q];
        if (stage_out) stage_out[q] = c_stage * kq + uq;
        acc_out[q] = c_acc * kq + a;
    }
}

// ---- FP64 issue-peak probes (register-only loops)
__global__ void k_probe_dmma(double *out, int iters, double a, double b) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = threadIdx.x * 1e-3 + i; c[i][1] = i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) dmma(c[i][0], c[i][1], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void k_probe_dfma(double *out, int iters, double a, double b) {
    double c[16];
#pragma unroll
    for (int i = 0; i < 16; i++) c[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) c[i] = fma(c[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += c[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
