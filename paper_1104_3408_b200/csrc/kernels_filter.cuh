// Yn tensor filter (eq. 51-56, 60-62):
//   k_project    dyad projection (eq. 54-56): Cartesian components -> spin-weight components ("dofs")
//   k_gemm_cols  phi analysis (eq. 33): real Fourier rows a_0, a_1, b_1, .., a_L, b_L of every dof
//   k_theta      per-(n,m) theta matrix F^n_m (eq. 62), complex components via c_{+-m} (reading Q12)
//   k_gemm_cols  phi synthesis (eq. 31)
//   k_recombine  recombination with the conjugate dyad (eq. 56), real part (eq. 60)
//
// The projection is done as a REAL rotation of every spatial index into the orthonormal frame
// (r^, theta^, phi^) of eq. (51) followed by the complex combinations of eq. (52):
//     contraction with m_a  = (V_theta + i V_phi)/sqrt2   -> spin weight +1 per index (reading Q7, App. B.3)
//     contraction with mbar = (V_theta - i V_phi)/sqrt2   -> spin weight -1
// For a real tensor the mbar<->m mirrored component is the complex conjugate and is not stored (eq. 50).
#pragma once
#include "sp_device.cuh"

enum { TT_SCALAR = 0, TT_VEC3, TT_VEC4, TT_SYM3, TT_SYM4, TT_R3_3_3, TT_R3_3_4, TT_R3_4_3, TT_R3_4_4, TT_COUNT };

#define SP_MAX_COMP 40
#define RSQRT2 0.70710678118654752440
#define SQRT2 1.41421356237309504880

struct Trig { double st, ct, sp, cp; };

__device__ __forceinline__ void rot3(const Trig &q, double x, double y, double z, double &vr, double &vt, double &vp) {
    const double a = q.cp * x + q.sp * y;
    vr = q.st * a + q.ct * z;
    vt = q.ct * a - q.st * z;
    vp = q.cp * y - q.sp * x;
}
__device__ __forceinline__ void irot3(const Trig &q, double vr, double vt, double vp, double &x, double &y, double &z) {
    const double a = q.st * vr + q.ct * vt;
    z = q.ct * vr - q.st * vt;
    x = q.cp * a - q.sp * vp;
    y = q.sp * a + q.cp * vp;
}

// symmetric D x D, canonical upper triangle.  D = 4: tt,t1,t2,t3,11,12,13,22,23,33; D = 3: 11,12,13,22,23,33.
template <int D> struct SymIdx { static constexpr int n = (D == 4) ? 10 : 6, o = (D == 4) ? 4 : 0; };

template <int D, bool INV>
__device__ __forceinline__ void rot_sym(const Trig &q, const double *S, double *R) {
    constexpr int o = SymIdx<D>::o;
    if (D == 4) {
        R[0] = S[0];
        if (INV) irot3(q, S[1], S[2], S[3], R[1], R[2], R[3]);
        else rot3(q, S[1], S[2], S[3], R[1], R[2], R[3]);
    }
    double T[3][3];   // T[a][B] = sum_b S[a][b] O[B][b]
    if (INV) {
        irot3(q, S[o + 0], S[o + 1], S[o + 2], T[0][0], T[0][1], T[0][2]);
        irot3(q, S[o + 1], S[o + 3], S[o + 4], T[1][0], T[1][1], T[1][2]);
        irot3(q, S[o + 2], S[o + 4], S[o + 5], T[2][0], T[2][1], T[2][2]);
    } else {
        rot3(q, S[o + 0], S[o + 1], S[o + 2], T[0][0], T[0][1], T[0][2]);
        rot3(q, S[o + 1], S[o + 3], S[o + 4], T[1][0], T[1][1], T[1][2]);
        rot3(q, S[o + 2], S[o + 4], S[o + 5], T[2][0], T[2][1], T[2][2]);
    }
    double c0[3], c1[3], c2[3];
    if (INV) {
        irot3(q, T[0][0], T[1][0], T[2][0], c0[0], c0[1], c0[2]);
        irot3(q, T[0][1], T[1][1], T[2][1], c1[0], c1[1], c1[2]);
        irot3(q, T[0][2], T[1][2], T[2][2], c2[0], c2[1], c2[2]);
    } else {
        rot3(q, T[0][0], T[1][0], T[2][0], c0[0], c0[1], c0[2]);
        rot3(q, T[0][1], T[1][1], T[2][1], c1[0], c1[1], c1[2]);
        rot3(q, T[0][2], T[1][2], T[2][2], c2[0], c2[1], c2[2]);
    }
    R[o + 0] = c0[0]; R[o + 1] = c1[0]; R[o + 2] = c2[0];
    R[o + 3] = c1[1]; R[o + 4] = c2[1]; R[o + 5] = c2[2];
}

// rotated symmetric block -> spin dofs.  D=4: [tt, tr, rr, mmbar | Re tm, Im tm, Re rm, Im rm, Re mm, Im mm]
// D=3: [rr, mmbar | Re rm, Im rm, Re mm, Im mm].   (indices of R: t,r,th,ph order)
template <int D>
__device__ __forceinline__ void sym_to_spin(const double *R, double *d) {
    constexpr int o = SymIdx<D>::o;
    int w = 0;
    if (D == 4) { d[w++] = R[0]; d[w++] = R[1]; }
    d[w++] = R[o + 0];                          // rr
    d[w++] = 0.5 * (R[o + 3] + R[o + 5]);       // m mbar = (thth + phph)/2
    if (D == 4) { d[w++] = RSQRT2 * R[2]; d[w++] = RSQRT2 * R[3]; }   // tm = (t th + i t ph)/sqrt2
    d[w++] = RSQRT2 * R[o + 1]; d[w++] = RSQRT2 * R[o + 2];          // rm
    d[w++] = 0.5 * (R[o + 3] - R[o + 5]); d[w++] = R[o + 4];         // mm = (thth - phph)/2 + i thph
}
template <int D>
__device__ __forceinline__ void spin_to_sym(const double *d, double *R) {
    constexpr int o = SymIdx<D>::o;
    int w = 0;
    if (D == 4) { R[0] = d[w++]; R[1] = d[w++]; }
    R[o + 0] = d[w++];
    const double mmb = d[w++];
    if (D == 4) { R[2] = SQRT2 * d[w++]; R[3] = SQRT2 * d[w++]; }
    R[o + 1] = SQRT2 * d[w++]; R[o + 2] = SQRT2 * d[w++];
    const double re = d[w++], im = d[w++];
    R[o + 3] = mmb + re; R[o + 5] = mmb - re; R[o + 4] = im;
}

// number of real dofs of the symmetric pattern that are real (n = 0) before the complex ones start
template <int D> struct SymPat { static constexpr int nreal = (D == 4) ? 4 : 2, ncplx = (D == 4) ? 3 : 2; };

struct TensorArgs {
    int field[SP_MAX_COMP];   // state field of stored component c
    int ncomp;
    int dof0;                 // first dof array of this tensor in the workspace
};

template <int TT> struct TTInfo;
template <> struct TTInfo<TT_SCALAR> { static constexpr int nc = 1; };
template <> struct TTInfo<TT_VEC3> { static constexpr int nc = 3; };
template <> struct TTInfo<TT_VEC4> { static constexpr int nc = 4; };
template <> struct TTInfo<TT_SYM3> { static constexpr int nc = 6; };
template <> struct TTInfo<TT_SYM4> { static constexpr int nc = 10; };
template <> struct TTInfo<TT_R3_3_3> { static constexpr int nc = 18; };
template <> struct TTInfo<TT_R3_3_4> { static constexpr int nc = 30; };
template <> struct TTInfo<TT_R3_4_3> { static constexpr int nc = 24; };
template <> struct TTInfo<TT_R3_4_4> { static constexpr int nc = 40; };

// rank 3, first index of dim D1, symmetric pair of dim D2.  dof order:
//   [A = t block (D1 = 4 only)] [A = r block]                         each the sym pattern (n as in sym)
//   [m ; real pattern entries]        complex, n = +1
//   [m ; complex pattern entries]     complex, n = n_e + 1
//   [mbar ; complex pattern entries]  complex, n = n_e - 1
template <int D1, int D2, bool INV>
__device__ __forceinline__ void r3_transform(const Trig &q, const double *in, double *out) {
    constexpr int ns = SymIdx<D2>::n, nr = SymPat<D2>::nreal, ncx = SymPat<D2>::ncplx, o1 = (D1 == 4) ? 1 : 0;
    double R[D1][ns];
    if (!INV) {
        double W[D1][ns];
#pragma unroll
        for (int a = 0; a < D1; a++) rot_sym<D2, false>(q, in + a * ns, W[a]);
#pragma unroll
        for (int e = 0; e < ns; e++) {
            if (D1 == 4) R[0][e] = W[0][e];
            rot3(q, W[o1 + 0][e], W[o1 + 1][e], W[o1 + 2][e], R[o1 + 0][e], R[o1 + 1][e], R[o1 + 2][e]);
        }
        int w = 0;
        if (D1 == 4) { sym_to_spin<D2>(R[0], out + w); w += ns; }
        sym_to_spin<D2>(R[o1], out + w); w += ns;
        double dt[ns], dp[ns];
        sym_to_spin<D2>(R[o1 + 1], dt);       // first index = theta
        sym_to_spin<D2>(R[o1 + 2], dp);       // first index = phi
#pragma unroll
        for (int e = 0; e < nr; e++) {        // [m; real e] = (e(th) + i e(ph))/sqrt2
            out[w++] = RSQRT2 * dt[e]; out[w++] = RSQRT2 * dp[e];
        }
#pragma unroll
        for (int e = 0; e < ncx; e++) {         // [m; c] = (c(th) + i c(ph))/sqrt2, c complex
            const double cr = dt[nr + 2 * e], ci = dt[nr + 2 * e + 1], er = dp[nr + 2 * e], ei = dp[nr + 2 * e + 1];
            out[w++] = RSQRT2 * (cr - ei); out[w++] = RSQRT2 * (ci + er);
        }
#pragma unroll
        for (int e = 0; e < ncx; e++) {         // [mbar; c] = (c(th) - i c(ph))/sqrt2
            const double cr = dt[nr + 2 * e], ci = dt[nr + 2 * e + 1], er = dp[nr + 2 * e], ei = dp[nr + 2 * e + 1];
            out[w++] = RSQRT2 * (cr + ei); out[w++] = RSQRT2 * (ci - er);
        }
    } else {
        int w = 0;
        if (D1 == 4) { spin_to_sym<D2>(in + w, R[0]); w += ns; }
        spin_to_sym<D2>(in + w, R[o1]); w += ns;
        double dt[ns], dp[ns];
#pragma unroll
        for (int e = 0; e < nr; e++) { dt[e] = SQRT2 * in[w++]; dp[e] = SQRT2 * in[w++]; }
        const double *pm = in + w, *pb = in + w + 2 * ncx;
#pragma unroll
        for (int e = 0; e < ncx; e++) {
            // X = (c_th + i c_ph)/sqrt2, Z = (c_th - i c_ph)/sqrt2  =>  c_th = (X+Z)/sqrt2, c_ph = (X-Z)/(i sqrt2)
            const double xr = pm[2 * e], xi = pm[2 * e + 1], zr = pb[2 * e], zi = pb[2 * e + 1];
            dt[nr + 2 * e] = RSQRT2 * (xr + zr); dt[nr + 2 * e + 1] = RSQRT2 * (xi + zi);
            dp[nr + 2 * e] = RSQRT2 * (xi - zi); dp[nr + 2 * e + 1] = -RSQRT2 * (xr - zr);
        }
        spin_to_sym<D2>(dt, R[o1 + 1]);
        spin_to_sym<D2>(dp, R[o1 + 2]);
        double W[D1][ns];
#pragma unroll
        for (int e = 0; e < ns; e++) {
            if (D1 == 4) W[0][e] = R[0][e];
            irot3(q, R[o1 + 0][e], R[o1 + 1][e], R[o1 + 2][e], W[o1 + 0][e], W[o1 + 1][e], W[o1 + 2][e]);
        }
#pragma unroll
        for (int a = 0; a < D1; a++) rot_sym<D2, true>(q, W[a], out + a * ns);
    }
}

template <int TT, bool INV>
__device__ __forceinline__ void tensor_transform(const Trig &q, const double *in, double *out) {
    if (TT == TT_SCALAR) {
        out[0] = in[0];
    } else if (TT == TT_VEC3 || TT == TT_VEC4) {
        constexpr int o = (TT == TT_VEC4) ? 1 : 0;
        if (TT == TT_VEC4) out[0] = in[0];
        if (!INV) {
            double vr, vt, vp;
            rot3(q, in[o], in[o + 1], in[o + 2], vr, vt, vp);
            out[o] = vr; out[o + 1] = RSQRT2 * vt; out[o + 2] = RSQRT2 * vp;   // m.v = (v_th + i v_ph)/sqrt2
        } else {
            irot3(q, in[o], SQRT2 * in[o + 1], SQRT2 * in[o + 2], out[o], out[o + 1], out[o + 2]);
        }
    } else if (TT == TT_SYM3 || TT == TT_SYM4) {
        constexpr int D = (TT == TT_SYM4) ? 4 : 3;
        double R[SymIdx<D>::n];
        if (!INV) { rot_sym<D, false>(q, in, R); sym_to_spin<D>(R, out); }
        else { spin_to_sym<D>(in, R); rot_sym<D, true>(q, R, out); }
    } else if (TT == TT_R3_3_3) r3_transform<3, 3, INV>(q, in, out);
    else if (TT == TT_R3_3_4) r3_transform<3, 4, INV>(q, in, out);
    else if (TT == TT_R3_4_3) r3_transform<4, 3, INV>(q, in, out);
    else if (TT == TT_R3_4_4) r3_transform<4, 4, INV>(q, in, out);
}

// pointwise: INV = false: state fields -> dof arrays; INV = true: dof arrays -> state fields
// pointwise, with the phi-reflection fold fused in.  The real Fourier transforms (eq. 20-24) see a function only
// through E_j = f_j + f_{J-j} (cosine rows) and O_j = f_j - f_{J-j} (sine rows), j = 1..J/2-1, plus f_0 and f_{J/2}:
//     a_m = (2/J) [ f_0 + (-1)^m f_{J/2} + sum_{j=1}^{J/2-1} cos(m phi_j) E_j ],   b_m = (2/J) sum_{j=1}^{J/2-1} sin(m phi_j) O_j,
// which halves the contraction length of the analysis and synthesis products (same sums, regrouped).
// Folded dof arrays [dof][row][i][k]: rows 0..J/2 hold f_0, E_1..E_{J/2-1}, f_{J/2}; rows J/2+j hold O_j.
// One thread owns the grid points (k, i, j) and (k, i, J-j), j = 0..J/2.
//   INV = false: state fields -> folded dofs;   INV = true: folded dofs -> state fields.
// tensors of the SAME index structure share one launch: blockIdx.y selects the tensor
#define SP_PW_GROUP 4
struct TensorArgsGroup { TensorArgs t[SP_PW_GROUP]; };

template <int TT, bool INV>
__global__ void __launch_bounds__(128)
k_pointwise(const __grid_constant__ TensorArgsGroup tg, int Nr, int Nt, size_t npts, const double *__restrict__ sin_t,
            const double *__restrict__ cos_t, const double *__restrict__ sin_p, const double *__restrict__ cos_p, const double *src,
            double *dst) {
    constexpr int nc = TTInfo<TT>::nc;
    const TensorArgs &ta = tg.t[blockIdx.y];
    const size_t plane = (size_t)Nr * Nt;
    const size_t q0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;       // (k, i, j) with j in [0, J/2]
    if (q0 >= plane * (size_t)(Nt + 1)) return;
    const int j = (int)(q0 / plane);
    const size_t ki = q0 - (size_t)j * plane;
    const int i = (int)(ki / Nr);
    const int J = 2 * Nt, j2 = J - j;
    const bool paired = (j != 0) && (j != Nt);
    const size_t p1 = (size_t)j * plane + ki, p2 = (size_t)j2 * plane + ki;   // the two grid points
    const size_t pe = p1, po = (size_t)(Nt + j) * plane + ki;                // folded rows E_j and O_j
    const double st = sin_t[i], ct = cos_t[i];
    const Trig t1 = {st, ct, sin_p[j], cos_p[j]};
    double a[nc], b[nc];
    if (!INV) {
        double in[nc];
#pragma unroll
        for (int c = 0; c < nc; c++) in[c] = src[(size_t)ta.field[c] * npts + p1];
        tensor_transform<TT, false>(t1, in, a);
        if (paired) {
            const Trig t2 = {st, ct, sin_p[j2], cos_p[j2]};
#pragma unroll
            for (int c = 0; c < nc; c++) in[c] = src[(size_t)ta.field[c] * npts + p2];
            tensor_transform<TT, false>(t2, in, b);
#pragma unroll
            for (int c = 0; c < nc; c++) {
                dst[(size_t)(ta.dof0 + c) * npts + pe] = a[c] + b[c];
                dst[(size_t)(ta.dof0 + c) * npts + po] = a[c] - b[c];
            }
        } else {
#pragma unroll
            for (int c = 0; c < nc; c++) dst[(size_t)(ta.dof0 + c) * npts + pe] = a[c];
        }
    } else {
        double out[nc];
        if (paired) {
#pragma unroll
            for (int c = 0; c < nc; c++) {
                const double e = src[(size_t)(ta.dof0 + c) * npts + pe], o = src[(size_t)(ta.dof0 + c) * npts + po];
                a[c] = e + o; b[c] = e - o;
            }
        } else {
#pragma unroll
            for (int c = 0; c < nc; c++) a[c] = src[(size_t)(ta.dof0 + c) * npts + pe];
        }
        tensor_transform<TT, true>(t1, a, out);
#pragma unroll
        for (int c = 0; c < nc; c++) dst[(size_t)ta.field[c] * npts + p1] = out[c];
        if (paired) {
            const Trig t2 = {st, ct, sin_p[j2], cos_p[j2]};
            tensor_transform<TT, true>(t2, b, out);
#pragma unroll
            for (int c = 0; c < nc; c++) dst[(size_t)ta.field[c] * npts + p2] = out[c];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// theta step (eq. 62).  coef[dof][mc][i][k], mc = m: a_m (m = 0..L); mc = L+m: b_m (m = 1..L).
// One CTA per (component, m); warp = column tile of 4 radii x {v = 0, 1} (columns interleaved
// col = 2k + v so that a lane's two accumulator columns are the (v=0, v=1) pair of one radius).
//   real component (n = 0):      a~_m = F^0_m a_m,  b~_m = F^0_m b_m
//   complex component g = gr + i gi of spin n (dofs d, d+1), m > 0:
//       Re c_m  = (a^r + b^i)/2, Im c_m  = (a^i - b^r)/2   -> F^n_m        -> (p, q)
//       Re c_-m = (a^r - b^i)/2, Im c_-m = (a^i + b^r)/2   -> F^{-n}_m     -> (s, t)   [F^n_{-m} = F^{-n}_m, eq. 47]
//       a~^r = p + s, b~^r = t - q, a~^i = q + t, b~^i = p - s
//     m = 0: a~^r_0 = F^n_0 a^r_0, a~^i_0 = F^n_0 a^i_0.
// Out of place (coef -> cout) so that row groups (blockIdx.z) and column tiles are independent.
// ---------------------------------------------------------------------------------------------
struct ThetaComp { int dof; int n; int cplx; };

#define SP_THETA_BATCH 64
struct ThetaBatch { ThetaComp c[SP_THETA_BATCH]; };

template <int MT>
__global__ void __launch_bounds__(32 * 20)
k_theta(ThetaBatch comps, const double *__restrict__ F, int L, int Nt, int Nt8, int Nt4, int Nr, int MC4,
        const double *__restrict__ coef, double *__restrict__ cout) {
    const ThetaComp cmp = comps.c[blockIdx.y];
    const int mt0 = blockIdx.z * MT;
    const int m = blockIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const size_t vec = (size_t)Nt * Nr;                       // one coefficient vector [i][k]
    const size_t dofsz = (size_t)MC4 * vec;
    const size_t fsz = (size_t)Nt8 * Nt4;
    if (4 * warp >= Nr) return;
    const int mca = m, mcb = L + m;                            // rows a_0..a_L, b_1..b_L
    const int kB = 4 * warp + (g >> 1), vB = g & 1;           // B-fragment column of this lane
    const bool kBok = kB < Nr;
    double acc1[MT][2], acc2[MT][2];
#pragma unroll
    for (int a = 0; a < MT; a++) acc1[a][0] = acc1[a][1] = acc2[a][0] = acc2[a][1] = 0.0;
    const int ksteps = (Nt + 3) >> 2;
    auto frag = [&](const double *Fm_, int mt, int ii) -> double {
        return (mt * 8 < Nt8) ? __ldg(Fm_ + (size_t)(mt * 8 + g) * Nt4 + ii) : 0.0;
    };

    if (!cmp.cplx) {
        const double *F0 = F + ((size_t)3 * (L + 1) + m) * fsz;
        const double *src = coef + (size_t)cmp.dof * dofsz + (size_t)(vB ? mcb : mca) * vec + kB;
        const bool ok = kBok && !(m == 0 && vB);
        for (int ks = 0; ks < ksteps; ks++) {
            const int ii = ks * 4 + t;
            const double bf = (ok && ii < Nt) ? src[(size_t)ii * Nr] : 0.0;
#pragma unroll
            for (int a = 0; a < MT; a++) dmma(acc1[a][0], acc1[a][1], frag(F0, mt0 + a, ii), bf);
        }
        const int k = 4 * warp + t;
        if (k < Nr) {
            double *da = cout + (size_t)cmp.dof * dofsz + (size_t)mca * vec + k;
            double *db = cout + (size_t)cmp.dof * dofsz + (size_t)mcb * vec + k;
#pragma unroll
            for (int a = 0; a < MT; a++) {
                const int i = (mt0 + a) * 8 + g;
                if (i < Nt) {
                    da[(size_t)i * Nr] = acc1[a][0];
                    if (m > 0) db[(size_t)i * Nr] = acc1[a][1];
                }
            }
        }
    } else {
        const double *Fp = F + ((size_t)(3 + cmp.n) * (L + 1) + m) * fsz;
        const double *Fm = F + ((size_t)(3 - cmp.n) * (L + 1) + m) * fsz;
        const double *R = coef + (size_t)cmp.dof * dofsz, *I = R + dofsz;
        double *Ro = cout + (size_t)cmp.dof * dofsz, *Io = Ro + dofsz;
        // v = 0: x = a^r, y = b^i;  v = 1: x = a^i, y = -b^r
        const double *px = (vB ? I : R) + (size_t)mca * vec + kB;
        const double *py = (vB ? R : I) + (size_t)mcb * vec + kB;
        const double ysgn = vB ? -1.0 : 1.0;
        for (int ks = 0; ks < ksteps; ks++) {
            const int ii = ks * 4 + t;
            double x = 0.0, y = 0.0;
            if (kBok && ii < Nt) {
                x = px[(size_t)ii * Nr];
                if (m > 0) y = ysgn * py[(size_t)ii * Nr];
            }
            const double b1 = (m > 0) ? 0.5 * (x + y) : x, b2 = 0.5 * (x - y);
#pragma unroll
            for (int a = 0; a < MT; a++) {
                dmma(acc1[a][0], acc1[a][1], frag(Fp, mt0 + a, ii), b1);
                if (m > 0) dmma(acc2[a][0], acc2[a][1], frag(Fm, mt0 + a, ii), b2);
            }
        }
        const int k = 4 * warp + t;
        if (k < Nr) {
#pragma unroll
            for (int a = 0; a < MT; a++) {
                const int i = (mt0 + a) * 8 + g;
                if (i < Nt) {
                    const double pp = acc1[a][0], qq = acc1[a][1], ss = acc2[a][0], tt = acc2[a][1];
                    const size_t off = (size_t)i * Nr + k;
                    if (m > 0) {
                        Ro[(size_t)mca * vec + off] = pp + ss;
                        Ro[(size_t)mcb * vec + off] = tt - qq;
                        Io[(size_t)mca * vec + off] = qq + tt;
                        Io[(size_t)mcb * vec + off] = pp - ss;
                    } else {
                        Ro[off] = pp;
                        Io[off] = qq;
                    }
                }
            }
        }
    }
}
