// Cartesian gradient (eq. 6; 142-166 eq. 13-19; 72 double cover).
//
//   sp_cartesian_gradient = k_gemm_cols<CIRC>  (d/dphi of every field, eq. 18 without transposes -> workspace)
//                         + k_grad_rtheta      (d/dr, d/dtheta on (r,theta) planes in shared memory, then the
//                                               chain rule (eq. 6) with d/dphi read back, writing d/dx, d/dy, d/dz)
#pragma once
#include "sp_device.cuh"

struct GradParams {
    int Nr, Nt, Np, PU, Nr8, Nr4, Nt8;
    const double *cd;       // [Nr8][PU]
    const double *g2;       // [2Nt]
    const double *inv_r, *sin_t, *cos_t, *inv_sin_t, *sin_p, *cos_p;
    const double *u;        // [nf] state
    const double *dphi;     // [nf] state (workspace)
    double *du;             // [3][nf] state
    int nf;
    int nitems;             // Nt * nf (field, plane-pair) work items of k_grad_rtheta2
};

// One CTA per (field mu, j < Nt): owns the antipodal pair of (r,theta) planes j and j+Nt
// (f(theta,phi) = f(2pi-theta, pi+phi)), so the double cover never touches memory.
// Shared memory: P[2][Nt8][PU] planes (row i, column k, zero padded), CDs[Nr8][PU], g2s[2Nt].
// Warp task = (plane, i-tile, group of KT k-tiles):
//   d/dtheta: C[i][k]  = sum_ii g2[(i-ii) mod 2Nt] * u_ext[ii][k]     A = circulant table, B = planes
//   d/dr    : C[i][k'] = sum_kk u[i][kk] * CD[k'][kk]                 A = plane rows,      B = CD^T
// Both leave the same C fragment (i = i0+g, k = k0+2t,+1), so the chain rule is lane-local.
template <int KT>
__global__ void __launch_bounds__(512) k_grad_rtheta(GradParams p) {
    extern __shared__ double sm[];
    const int Nr = p.Nr, Nt = p.Nt, Np = p.Np, PU = p.PU;
    double *P0 = sm, *P1 = sm + (size_t)p.Nt8 * PU, *CDs = P1 + (size_t)p.Nt8 * PU, *g2s = CDs + (size_t)p.Nr8 * PU;
    const int j = blockIdx.x, mu = blockIdx.y;
    const size_t npts = (size_t)Nr * Nt * Np, plane = (size_t)Nr * Nt;
    const double *u0 = p.u + mu * npts + (size_t)j * plane, *u1 = u0 + (size_t)Nt * plane;

    for (int q = threadIdx.x; q < 2 * p.Nt8 * PU; q += blockDim.x) sm[q] = 0.0;
    for (int q = threadIdx.x; q < p.Nr8 * PU; q += blockDim.x) CDs[q] = p.cd[q];
    for (int q = threadIdx.x; q < 2 * Nt; q += blockDim.x) g2s[q] = p.g2[q];
    __syncthreads();
    for (int q = threadIdx.x; q < Nt * Nr; q += blockDim.x) {
        const int i = q / Nr, k = q - i * Nr;
        P0[i * PU + k] = u0[q];
        P1[i * PU + k] = u1[q];
    }
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int itiles = p.Nt8 >> 3, ktiles = p.Nr8 >> 3, kgroups = (ktiles + KT - 1) / KT;
    const int ntasks = 2 * itiles * kgroups;
    const int n2 = 2 * Nt;
    for (int task = warp; task < ntasks; task += nwarps) {
        const int pl = task / (itiles * kgroups);
        const int rem = task - pl * itiles * kgroups;
        const int it = rem / kgroups, kg = rem - it * kgroups;
        const double *Pown = pl ? P1 : P0, *Poth = pl ? P0 : P1;
        const int i0 = it * 8, kt0 = kg * KT;
        double at[KT][2], ar[KT][2];
#pragma unroll
        for (int q = 0; q < KT; q++) at[q][0] = at[q][1] = ar[q][0] = ar[q][1] = 0.0;
        // ---- d/dtheta: K = 2Nt over the extended latitude index ii
        const int irow = i0 + g;
        for (int ks = 0; ks < (n2 + 3) / 4; ks++) {
            const int ii = ks * 4 + t;
            int d = irow - ii;
            d += (d < 0) ? n2 : 0;
            const double af = (ii < n2 && irow < Nt) ? g2s[d] : 0.0;
            const int iic = ii < n2 ? ii : n2 - 1;
            const double *rowp = (iic < Nt) ? (Pown + iic * PU) : (Poth + (n2 - 1 - iic) * PU);
#pragma unroll
            for (int q = 0; q < KT; q++) {
                const int kc = (kt0 + q) * 8 + g;
                const double bf = (kt0 + q < ktiles) ? rowp[kc] : 0.0;
                dmma(at[q][0], at[q][1], af, bf);
            }
        }
        // ---- d/dr: K = Nr over kk;  A = u[i0+g][kk], B[kk][k'] = CD[k'][kk]
        for (int ks = 0; ks < p.Nr4 / 4; ks++) {
            const int kk = ks * 4 + t;
            const double af = Pown[irow * PU + kk];
#pragma unroll
            for (int q = 0; q < KT; q++) {
                const int kp = (kt0 + q) * 8 + g;
                const double bf = (kt0 + q < ktiles) ? CDs[kp * PU + kk] : 0.0;
                dmma(ar[q][0], ar[q][1], af, bf);
            }
        }
        // ---- chain rule (eq. 6), lane-local
        if (irow < Nt) {
            const int jj = pl ? j + Nt : j;
            const double st = p.sin_t[irow], ct = p.cos_t[irow], ist = p.inv_sin_t[irow];
            const double sp = p.sin_p[jj], cp = p.cos_p[jj];
            const size_t base = (size_t)mu * npts + (size_t)jj * plane + (size_t)irow * Nr;
            const size_t fs = (size_t)p.nf * npts;
#pragma unroll
            for (int q = 0; q < KT; q++) {
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const int k = (kt0 + q) * 8 + 2 * t + e;
                    if (k < Nr) {
                        const double ir = p.inv_r[k];
                        const double a = ar[q][e], b = at[q][e] * ir, c = p.dphi[base + k] * ir * ist;
                        p.du[base + k] = st * cp * a + ct * cp * b - sp * c;
                        p.du[fs + base + k] = st * sp * a + ct * sp * b + cp * c;
                        p.du[2 * fs + base + k] = ct * a - st * b;
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// v2 of the (r,theta)-plane kernel: same mathematics and data flow as k_grad_rtheta, but
//   * warp task = (plane, PAIR of latitude tiles, group of 3 radial tiles): every A fragment feeds 3 and
//     every B fragment 2 DMMAs (0.83 shared-memory loads per DMMA instead of 1.2);
//   * <= 85 registers so that two CTAs share an SM and one CTA's plane load / epilogue overlaps the
//     other's tensor work; planes arrive by 8-byte cp.async while the CD^ table is copied;
//   * only the padding (columns >= Nr, rows >= Nt) is zero-filled.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async8g(void *smem, const void *gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gmem));
}

// Preconditions (checked by the launcher, else the generic k_grad_rtheta runs): Ntheta % 4 == 0.
// Layout of shared memory: P0, P1 [Nt8][PU] (PU >= padded column count, = 4 mod 8), CDs [NK8][PU] with
// NK8 = kgroups*KT*8 rows, g2d [4 Nt + 8] = the circulant generator of FD_{2Nt} repeated twice.
// Garbage in padded ROWS / COLUMNS of an operand only reaches discarded outputs (DMMA rows and columns are
// independent); only the contraction padding (kk >= Nr) must be zero, and it is, in both operands.
// SPLIT = true: the kernel runs FIRST and writes the phi-independent combinations
//     W = sin(th) d_r u + (cos(th)/r) d_th u  -> du[0] (x slot),     d_z u = cos(th) d_r u - (sin(th)/r) d_th u -> du[2];
// the d/dphi GEMM that follows (k_phi_gemm<.., EPI_GRAD>) finishes d_x = cos(ph) W - sin(ph) c, d_y = sin(ph) W + cos(ph) c
// with c = d_phi u /(r sin th) in its epilogue.  No global read sits on this kernel's critical path.
// SPLIT = false: d/dphi is read from p.dphi and all three components are finished here.
// PERSISTENT: each CTA walks the work items (field mu, plane pair j) it = blockIdx.x, blockIdx.x + gridDim.x, ...
// The CD^ / circulant / Jacobian tables are loaded once per CTA.  With NBUF = 2 the planes of the NEXT item stream into
// the other buffer (cp.async) while the tensor work of the current item runs, and the stores of the previous item drain
// meanwhile: measured with %globaltimer, the non-persistent version spent 3.5 us loading + 4 us storing per 8.6 us of
// DMMA work, all CTAs of a wave in lock-step (memory system and tensor pipes taking turns).
template <int KT, bool SPLIT, int NBUF>
__global__ void __launch_bounds__(KT == 3 ? 384 : 192, KT == 3 ? 1 : 2) k_grad_rtheta2(GradParams p) {
    extern __shared__ double sm[];
    const int Nr = p.Nr, Nt = p.Nt, Np = p.Np, PU = p.PU;
    const int itiles = p.Nt8 >> 3, ipairs = (itiles + 1) >> 1, ktiles = p.Nr8 >> 3, kgroups = (ktiles + KT - 1) / KT;
    const int NK8 = kgroups * KT * 8, n2 = 2 * Nt;
    const int prow = p.Nt8 + ((itiles & 1) ? 8 : 0);           // rows of a plane buffer
    const size_t planesz = (size_t)prow * PU;
    double *CDs = sm, *g2d = CDs + (size_t)NK8 * PU;
    double *tir = g2d + 2 * n2 + 8, *tst = tir + NK8, *tct = tst + p.Nt8 + 8, *tis = tct + p.Nt8 + 8;   // 1/r, sin, cos, 1/sin(theta)
    double *Pbuf = tis + p.Nt8 + 8;                                                                     // NBUF x [P0, P1]
    const size_t npts = (size_t)Nr * Nt * Np, plane = (size_t)Nr * Nt;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;

    // planes of one item: one latitude row per warp iteration, 8-byte cp.async into the padded pitch
    auto issue_planes = [&](int it, double *B0) {
        const int mu_ = it / Nt, j_ = it - mu_ * Nt;
        const double *u0 = p.u + mu_ * npts + (size_t)j_ * plane, *u1 = u0 + (size_t)Nt * plane;
        double *B1 = B0 + planesz;
        for (int i = warp; i < Nt; i += nwarps)
            for (int k = lane; k < Nr; k += 32) {
                cp_async8g(B0 + i * PU + k, u0 + (size_t)i * Nr + k);
                cp_async8g(B1 + i * PU + k, u1 + (size_t)i * Nr + k);
            }
    };
    // padding (columns >= Nr, rows >= Nt) of every buffer: zero, once
    for (int bq = 0; bq < 2 * NBUF; bq++) {
        double *B = Pbuf + bq * planesz;
        for (int i = warp; i < prow; i += nwarps)
            for (int k = lane; k < PU; k += 32)
                if (!(i < Nt && k < Nr)) B[i * PU + k] = 0.0;
    }
    // CD^ rows (16-byte copies: the pitch PU is even), circulant table and Jacobian tables: all asynchronous
    for (int q = threadIdx.x; q < NK8 * (PU / 2); q += blockDim.x) {
        const int r = q / (PU / 2), h = q - r * (PU / 2);
        if (r < p.Nr8) {
            unsigned sa = (unsigned)__cvta_generic_to_shared(CDs + r * PU + 2 * h);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(p.cd + r * PU + 2 * h));
        } else {
            CDs[r * PU + 2 * h] = 0.0; CDs[r * PU + 2 * h + 1] = 0.0;
        }
    }
    for (int q = threadIdx.x; q < 2 * n2 + 8; q += blockDim.x) cp_async8g(g2d + q, p.g2 + (q % n2));
    for (int q = threadIdx.x; q < NK8; q += blockDim.x) {
        if (q < Nr) cp_async8g(tir + q, p.inv_r + q); else tir[q] = 0.0;
    }
    for (int q = threadIdx.x; q < p.Nt8 + 8; q += blockDim.x) {
        if (q < Nt) { cp_async8g(tst + q, p.sin_t + q); cp_async8g(tct + q, p.cos_t + q); cp_async8g(tis + q, p.inv_sin_t + q); }
        else { tst[q] = 0.0; tct[q] = 0.0; tis[q] = 0.0; }
    }
    if ((int)blockIdx.x < p.nitems) issue_planes(blockIdx.x, Pbuf);
    asm volatile("cp.async.commit_group;\n" ::);

    const int g = lane >> 2, t = lane & 3;
    const int ntasks = 2 * ipairs * kgroups;
  int nloc = 0;
  for (int it = blockIdx.x; it < p.nitems; it += gridDim.x, nloc++) {
    const int mu = it / Nt, j = it - mu * Nt;
    double *P0 = Pbuf + (size_t)(NBUF == 2 ? (nloc & 1) : 0) * 2 * planesz, *P1 = P0 + planesz;
    if (NBUF == 2) {
        const int nxt = it + gridDim.x;
        if (nxt < p.nitems) issue_planes(nxt, Pbuf + (size_t)((nloc + 1) & 1) * 2 * planesz);
        asm volatile("cp.async.commit_group;\n" ::);
        asm volatile("cp.async.wait_group 1;\n" ::);
    } else {
        asm volatile("cp.async.wait_group 0;\n" ::);
    }
    __syncthreads();
    for (int task = warp; task < ntasks; task += nwarps) {
        const int pl = task / (ipairs * kgroups);
        const int rem = task - pl * ipairs * kgroups;
        const int ip = rem / kgroups, kg = rem - ip * kgroups;
        const double *Pown = pl ? P1 : P0, *Poth = pl ? P0 : P1;
        const int kt0 = kg * KT;
        const int ir0 = ip * 16 + g, ir1 = ir0 + 8;          // the lane's two latitude rows (rows < Nt8 + 8 exist)
        double at[2][KT][2], ar[2][KT][2];
#pragma unroll
        for (int a = 0; a < 2; a++)
#pragma unroll
            for (int q = 0; q < KT; q++) at[a][q][0] = at[a][q][1] = ar[a][q][0] = ar[a][q][1] = 0.0;
        // ---- d/dtheta (eq. 8 on the double cover): A[i][ii] = g2[(i - ii) mod 2Nt]
        //      first half ii < Nt: rows of the own plane ascending; second half: rows of the antipodal plane descending
        {
            const double *ga0 = g2d + (ir0 - t + n2), *ga1 = ga0 + 8;      // index (i - ii) + 2Nt, ii = 4 ks + t
            const double *bp = Pown + t * PU + kt0 * 8 + g;
#pragma unroll 2
            for (int ks = 0; ks < Nt / 4; ks++) {
                const double a0 = ga0[-4 * ks], a1 = ga1[-4 * ks];
#pragma unroll
                for (int q = 0; q < KT; q++) {
                    const double bf = bp[(size_t)ks * 4 * PU + q * 8];
                    dmma(at[0][q][0], at[0][q][1], a0, bf);
                    dmma(at[1][q][0], at[1][q][1], a1, bf);
                }
            }
            ga0 -= Nt; ga1 -= Nt;
            bp = Poth + (Nt - 1 - t) * PU + kt0 * 8 + g;                    // ii = Nt + 4 ks + t  ->  row 2Nt-1-ii
#pragma unroll 2
            for (int ks = 0; ks < Nt / 4; ks++) {
                const double a0 = ga0[-4 * ks], a1 = ga1[-4 * ks];
#pragma unroll
                for (int q = 0; q < KT; q++) {
                    const double bf = bp[-(ptrdiff_t)ks * 4 * PU + q * 8];
                    dmma(at[0][q][0], at[0][q][1], a0, bf);
                    dmma(at[1][q][0], at[1][q][1], a1, bf);
                }
            }
        }
        // d/dphi of the lane's outputs: prefetched into L1 now, read after the d/dr loop (hides the global latency)
        const int jj = pl ? j + Nt : j;
        const size_t pbase = (size_t)mu * npts + (size_t)jj * plane;
#pragma unroll
        for (int a = 0; a < 2; a++) {
            const int irow = a ? ir1 : ir0;
#pragma unroll
            for (int q = 0; q < KT; q++) {
                const int k = (kt0 + q) * 8 + 2 * t;
                if (!SPLIT && irow < Nt && k < Nr) asm volatile("prefetch.global.L1 [%0];\n" ::"l"(p.dphi + pbase + (size_t)irow * Nr + k));
            }
        }
        const double sp = SPLIT ? 0.0 : __ldg(p.sin_p + jj), cp = SPLIT ? 1.0 : __ldg(p.cos_p + jj);
        // ---- d/dr: A = u[i][kk], B[kk][k'] = CD^[k'][kk]   (eq. 9, 13)
        {
            const double *arow0 = Pown + ir0 * PU + t, *arow1 = arow0 + 8 * PU;
            const double *cdp = CDs + (kt0 * 8 + g) * PU + t;
#pragma unroll 3
            for (int ks = 0; ks < p.Nr4 / 4; ks++) {
                const double a0 = arow0[ks * 4], a1 = arow1[ks * 4];
#pragma unroll
                for (int q = 0; q < KT; q++) {
                    const double bf = cdp[q * 8 * PU + ks * 4];
                    dmma(ar[0][q][0], ar[0][q][1], a0, bf);
                    dmma(ar[1][q][0], ar[1][q][1], a1, bf);
                }
            }
        }
        // ---- chain rule (eq. 6), lane-local
        const size_t fs = (size_t)p.nf * npts;
#pragma unroll
        for (int a = 0; a < 2; a++) {
            const int irow = a ? ir1 : ir0;
            if (irow >= Nt) continue;
            const double st = tst[irow], ct = tct[irow], ist = tis[irow];
            const double xa = st * cp, xb = ct * cp, ya = st * sp, yb = ct * sp;
            const size_t base = pbase + (size_t)irow * Nr;
#pragma unroll
            for (int q = 0; q < KT; q++) {
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const int k = (kt0 + q) * 8 + 2 * t + e;
                    if (k < Nr) {
                        const double ir = tir[k];
                        const double va = ar[a][q][e], vb = at[a][q][e] * ir;
                        if (SPLIT) {
                            p.du[base + k] = st * va + ct * vb;
                            p.du[2 * fs + base + k] = ct * va - st * vb;
                        } else {
                            const double vc = __ldg(p.dphi + base + k) * (ir * ist);
                            p.du[base + k] = xa * va + xb * vb - sp * vc;
                            p.du[fs + base + k] = ya * va + yb * vb + cp * vc;
                            p.du[2 * fs + base + k] = ct * va - st * vb;
                        }
                    }
                }
            }
        }
    }
    __syncthreads();                       // every warp is done with this item's planes
    if (NBUF == 1) {
        const int nxt = it + gridDim.x;
        if (nxt < p.nitems) issue_planes(nxt, Pbuf);
        asm volatile("cp.async.commit_group;\n" ::);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// v3: as k_grad_rtheta2<.., SPLIT = true, ..> plus the REFLECTION FOLD of the theta derivative.  FD_{2Ntheta} is an
// antisymmetric circulant and the double cover is [own plane ascending | antipodal plane descending], so with
// E = (P_j + P_{j+Ntheta})/2, O = (P_j - P_{j+Ntheta})/2 (formed in shared memory)
//     d_theta P_j = G+ E + G- O,   d_theta P_{j+Ntheta} = G+ E - G- O,   G+-[i][r] = g(i - r) +- g(i + r + 1),
// two Ntheta x Ntheta products instead of two Ntheta x 2Ntheta ones: the same sums regrouped, half the DMMAs.  d/dr is
// linear, so it is taken on E and O as well and the planes are unfolded in the lane-local epilogue.
// Warp task = (latitude tile, group of KT radial tiles), four accumulator sets (theta/r x E/O).
// ---------------------------------------------------------------------------------------------
// PUC > 0: the shared-memory pitch as a compile-time constant (the pitches of the BASELINE configurations are instantiated), so
// that the fragment addresses of the two product loops fold into immediates; PUC = 0: pitch from the arguments.
template <int KT, int NBUF, int PUC = 0>
__global__ void __launch_bounds__(KT == 3 ? 384 : 192, KT == 3 ? 1 : 2) k_grad_rtheta3(GradParams p) {
    extern __shared__ double sm[];
    const int Nr = p.Nr, Nt = p.Nt, Np = p.Np, PU = PUC > 0 ? PUC : p.PU;
    const int itiles = p.Nt8 >> 3, ktiles = p.Nr8 >> 3, kgroups = (ktiles + KT - 1) / KT;
    const int NK8 = kgroups * KT * 8, n2 = 2 * Nt;
    const int prow = p.Nt8 + ((itiles & 1) ? 8 : 0);           // rows of a plane buffer
    const size_t planesz = (size_t)prow * PU;
    double *CDs = sm, *g2d = CDs + (size_t)NK8 * PU;
    double *tir = g2d + 2 * n2 + 8, *tst = tir + NK8, *tct = tst + p.Nt8 + 8, *tis = tct + p.Nt8 + 8;   // 1/r, sin, cos, 1/sin(theta)
    double *Pbuf = tis + p.Nt8 + 8;                                                                     // NBUF x [P0, P1]
    const size_t npts = (size_t)Nr * Nt * Np, plane = (size_t)Nr * Nt;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;

    // planes of one item: a plane is Nr*Nt contiguous doubles in global memory; thread e, e + blockDim, .. copies element e
    // (8-byte cp.async, coalesced) to row i = e / Nr, column k = e % Nr of the padded pitch.  (i, k) advance incrementally: the
    // loader's instruction count matters as much as the tensor loop's (it was 19 % of the kernel's instructions as a nested
    // row / column loop)
    const int ldi = blockDim.x / Nr, ldk = blockDim.x - ldi * Nr, lstep = ldi * PU + ldk;
    const int li0 = threadIdx.x / Nr, lk0 = threadIdx.x - li0 * Nr, nplane = Nr * Nt;
    auto issue_planes = [&](int it, double *B0) {
        const int mu_ = it / Nt, j_ = it - mu_ * Nt;
        const double *u0 = p.u + mu_ * npts + (size_t)j_ * plane + threadIdx.x, *u1 = u0 + (size_t)Nt * plane;
        double *s0 = B0 + li0 * PU + lk0, *s1 = s0 + planesz;
        int k = lk0;
#pragma unroll 1
        for (int e = threadIdx.x; e < nplane; e += blockDim.x) {
            cp_async8g(s0, u0);
            cp_async8g(s1, u1);
            u0 += blockDim.x; u1 += blockDim.x; k += ldk; s0 += lstep; s1 += lstep;
            if (k >= Nr) { k -= Nr; s0 += PU - Nr; s1 += PU - Nr; }
        }
    };
    // padding (columns >= Nr, rows >= Nt) of every buffer: zero, once
    for (int bq = 0; bq < 2 * NBUF; bq++) {
        double *B = Pbuf + bq * planesz;
        for (int i = warp; i < prow; i += nwarps)
            for (int k = lane; k < PU; k += 32)
                if (!(i < Nt && k < Nr)) B[i * PU + k] = 0.0;
    }
    // CD^ rows (16-byte copies: the pitch PU is even), circulant table and Jacobian tables: all asynchronous
    for (int q = threadIdx.x; q < NK8 * (PU / 2); q += blockDim.x) {
        const int r = q / (PU / 2), h = q - r * (PU / 2);
        if (r < p.Nr8) {
            unsigned sa = (unsigned)__cvta_generic_to_shared(CDs + r * PU + 2 * h);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(p.cd + r * PU + 2 * h));
        } else {
            CDs[r * PU + 2 * h] = 0.0; CDs[r * PU + 2 * h + 1] = 0.0;
        }
    }
    for (int q = threadIdx.x; q < 2 * n2 + 8; q += blockDim.x) cp_async8g(g2d + q, p.g2 + (q % n2));
    for (int q = threadIdx.x; q < NK8; q += blockDim.x) {
        if (q < Nr) cp_async8g(tir + q, p.inv_r + q); else tir[q] = 0.0;
    }
    for (int q = threadIdx.x; q < p.Nt8 + 8; q += blockDim.x) {
        if (q < Nt) { cp_async8g(tst + q, p.sin_t + q); cp_async8g(tct + q, p.cos_t + q); cp_async8g(tis + q, p.inv_sin_t + q); }
        else { tst[q] = 0.0; tct[q] = 0.0; tis[q] = 0.0; }
    }
    if ((int)blockIdx.x < p.nitems) issue_planes(blockIdx.x, Pbuf);
    asm volatile("cp.async.commit_group;\n" ::);

    const int g = lane >> 2, t = lane & 3;
    const int ntasks = itiles * kgroups;
  int nloc = 0;
  for (int it = blockIdx.x; it < p.nitems; it += gridDim.x, nloc++) {
    const int mu = it / Nt, j = it - mu * Nt;
    double *P0 = Pbuf + (size_t)(NBUF == 2 ? (nloc & 1) : 0) * 2 * planesz, *P1 = P0 + planesz;
    if (NBUF == 2) {
        const int nxt = it + gridDim.x;
        if (nxt < p.nitems) issue_planes(nxt, Pbuf + (size_t)((nloc + 1) & 1) * 2 * planesz);
        asm volatile("cp.async.commit_group;\n" ::);
        asm volatile("cp.async.wait_group 1;\n" ::);
    } else {
        asm volatile("cp.async.wait_group 0;\n" ::);
    }
    __syncthreads();
    // fold: E = (P0 + P1)/2, O = (P0 - P1)/2 in place (valid region; the padding stays zero)
    {   // flat over the first Nt rows, two doubles per thread and step (the pitch PU is even)
        double2 *A2 = reinterpret_cast<double2 *>(P0), *B2 = reinterpret_cast<double2 *>(P1);
        const int n2v = Nt * PU / 2;
#pragma unroll 4
        for (int q = threadIdx.x; q < n2v; q += blockDim.x) {
            const double2 x = A2[q], y = B2[q];
            A2[q] = make_double2(0.5 * (x.x + y.x), 0.5 * (x.y + y.y));
            B2[q] = make_double2(0.5 * (x.x - y.x), 0.5 * (x.y - y.y));
        }
    }
    __syncthreads();
    if (NBUF == 1 && threadIdx.x < 2) {
        // single-buffered (the plane pair of a large grid fills the SM's shared memory): the next item's planes cannot be staged
        // under this item's products, but they can be pulled into L2 (one bulk prefetch per plane: a plane is Nr*Ntheta contiguous
        // doubles), so that the exposed load phase of the next iteration reads L2 instead of HBM
        const int nxt = it + gridDim.x;
        if (nxt < p.nitems && !((nplane * 8) & 15)) {
            const int mu_ = nxt / Nt, j_ = nxt - mu_ * Nt;
            const double *up = p.u + mu_ * npts + (size_t)(j_ + (threadIdx.x ? Nt : 0)) * plane;
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(up), "r"(nplane * 8) : "memory");
        }
    }
    for (int task = warp; task < ntasks; task += nwarps) {
        const int it_ = task / kgroups, kg = task - it_ * kgroups;
        const int kt0 = kg * KT;
        const int ir0 = it_ * 8 + g;                              // the lane's latitude row
        double tE[KT][2], tO[KT][2], rE[KT][2], rO[KT][2];
#pragma unroll
        for (int q = 0; q < KT; q++) tE[q][0] = tE[q][1] = tO[q][0] = tO[q][1] = rE[q][0] = rE[q][1] = rO[q][0] = rO[q][1] = 0.0;
        // ---- d/dtheta on the folded planes: Gp/m[i][r] = g(i - r) +/- g(i + r + 1), K = Ntheta
        {
            const double *ga = g2d + (ir0 - t + n2), *gb = g2d + (ir0 + t + 1);
            const double *bE = P0 + t * PU + kt0 * 8 + g, *bO = P1 + t * PU + kt0 * 8 + g;
#pragma unroll 2
            for (int ks = 0; ks < Nt / 4; ks++) {
                const double x = ga[-4 * ks], y = gb[4 * ks];
                const double ap = x + y, am = x - y;
#pragma unroll
                for (int q = 0; q < KT; q++) {
                    dmma(tE[q][0], tE[q][1], ap, bE[(size_t)ks * 4 * PU + q * 8]);
                    dmma(tO[q][0], tO[q][1], am, bO[(size_t)ks * 4 * PU + q * 8]);
                }
            }
        }
        // ---- d/dr on E and O: A = plane rows, B[kk][k'] = CD^[k'][kk]   (eq. 9, 13)
        {
            const double *aE = P0 + ir0 * PU + t, *aO = P1 + ir0 * PU + t;
            const double *cdp = CDs + (kt0 * 8 + g) * PU + t;
#pragma unroll 3
            for (int ks = 0; ks < p.Nr4 / 4; ks++) {
                const double a0 = aE[ks * 4], a1 = aO[ks * 4];
#pragma unroll
                for (int q = 0; q < KT; q++) {
                    const double bf = cdp[q * 8 * PU + ks * 4];
                    dmma(rE[q][0], rE[q][1], a0, bf);
                    dmma(rO[q][0], rO[q][1], a1, bf);
                }
            }
        }
        // ---- unfold (plane j: E + O, plane j + Ntheta: E - O) and the phi-independent part of the chain rule (eq. 6)
        if (ir0 < Nt) {
            const double st = tst[ir0], ct = tct[ir0];
            const size_t fs = (size_t)p.nf * npts;
            const size_t b0 = (size_t)mu * npts + (size_t)j * plane + (size_t)ir0 * Nr, b1 = b0 + (size_t)Nt * plane;
#pragma unroll
            for (int q = 0; q < KT; q++) {
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const int k = (kt0 + q) * 8 + 2 * t + e;
                    if (k < Nr) {
                        const double ir = tir[k];
                        const double r0 = rE[q][e] + rO[q][e], r1 = rE[q][e] - rO[q][e];
                        const double t0 = (tE[q][e] + tO[q][e]) * ir, t1 = (tE[q][e] - tO[q][e]) * ir;
                        p.du[b0 + k] = st * r0 + ct * t0;
                        p.du[2 * fs + b0 + k] = ct * r0 - st * t0;
                        p.du[b1 + k] = st * r1 + ct * t1;
                        p.du[2 * fs + b1 + k] = ct * r1 - st * t1;
                    }
                }
            }
        }
    }
    __syncthreads();                       // every warp is done with this item's planes
    if (NBUF == 1) {
        const int nxt = it + gridDim.x;
        if (nxt < p.nitems) issue_planes(nxt, Pbuf);
        asm volatile("cp.async.commit_group;\n" ::);
    }
  }
}

// shared memory of k_grad_rtheta2<KT>
static inline size_t grad2_smem_bytes(int Nt, int Nt8, int Nr8, int PU, int KT, int nbuf, int nwarps) {
    const int ktiles = Nr8 / 8, NK8 = ((ktiles + KT - 1) / KT) * KT * 8, itiles = Nt8 / 8;
    const int prow = Nt8 + ((itiles & 1) ? 8 : 0);
    return ((size_t)nbuf * 2 * prow * PU + (size_t)NK8 * PU + 4 * Nt + 8 + NK8 + 3 * (Nt8 + 8)) * sizeof(double);
}
