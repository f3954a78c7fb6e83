// phi-direction contraction, shared-memory staged (the hot GEMM: d/dphi, phi analysis, phi synthesis).
//     C[b][m][c] = sum_k A[m][k] * B[b][k][c],   B[b][k][c] = B + b*sBb + k*sBk + c  (columns contiguous)
// (eq. 17-19 without the transposes; 254-259 eq. 33; 243-246 eq. 31.)
// CTA tile = ALL rows of A x NC columns (NC = 64; 32 when the 64-wide grid would leave SMs idle or with a single CTA: small
// states, see phi_ncol); K walked in chunks of 16 through a 3-stage cp.async pipeline:
//   As[stage][Mpad][20]    (pitch 20 doubles: fragment reads hit 16 distinct 8-byte banks)
//   Bs[stage][16][NC + 4]  (pitch = 4 mod 16: likewise)
// Warp (mg, ng): MT m-tiles x 2 n-tiles of 8x8, DMMA.8x8x4; NC/16 warps along the columns.  Requires even strides / ncols and 16-byte
// aligned bases (checked by the launcher; otherwise the generic kernel of kernels_gemm.cuh is used).
#pragma once
#include "sp_device.cuh"

#include <cstdint>
#include <cstdlib>
#include <algorithm>

// launches whose row blocks share an operand larger than this put the row-block index first in launch order
#define SP_SPLIT_FAST_BYTES (32.0 * 1024 * 1024)
#define PG_NCOL 64
#define PG_KC 16
#define PG_STAGES 3
#define PG_PA 20

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
// 16-byte cp.async; with ignore = true the source is not read and zeros are written
__device__ __forceinline__ void cp_async16_ign(void *smem, const void *gmem, bool ignore) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %2, 0;\n cp.async.cg.shared.global [%0], [%1], 16, p;\n}\n" ::"r"(s), "l"(gmem), "r"((int)ignore));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// EPI_GRAD: gradient epilogue (eq. 6).  The product is d/dphi u (A = FD_{Nphi}); C holds on entry the
// phi-independent combination W written by k_grad_rtheta3 and receives d_x u; Y receives d_y u:
//     c = (d_phi u)/(r sin th),   d_x = cos(ph) W - sin(ph) c,   d_y = sin(ph) W + cos(ph) c.
// Two-phase epilogue: c is parked in shared memory (the pipeline buffers are free by then), then all threads walk the tile
// row-contiguously with coalesced 16-byte loads of W and stores of d_x, d_y.
struct PhiGradEpi {
    double *Y; long sYb;                      // d_y output, batch stride
    const double *inv_r, *inv_sin_t, *sin_p, *cos_p;
    int Nr;
};

template <int MT, bool EPI_GRAD, int NC>
__global__ void __launch_bounds__(NC * 8)
k_phi_gemm(const double *__restrict__ A, int lda, int M, int Mpad, int K, const double *__restrict__ B, long sBk, long sBb,
           double *__restrict__ C, long sCm, long sCb, int ncols, PhiGradEpi ge, int sfast) {
    extern __shared__ __align__(16) double sm[];
    // grid = (column tiles, batch, row blocks), or with sfast (row blocks, column tiles, batch): the row blocks of one column tile
    // read the same B columns; as neighbours in launch order (x fastest) the second one finds them in L2 instead of DRAM.  That pays
    // when B is larger than L2 can keep; for small launches the simultaneous hits on the same lines cost more than they save.
    const int nzs = sfast ? gridDim.x : gridDim.z, bz = sfast ? blockIdx.x : blockIdx.z;
    const int bx = sfast ? blockIdx.y : blockIdx.x, by = sfast ? blockIdx.z : blockIdx.y;
    if (nzs > 1) {                                // row blocks: this CTA owns rows [r0, r0 + Mpad / gridDim.x)
        Mpad /= nzs;
        const int r0 = bz * Mpad;
        M = min(M - r0, Mpad);
        A += (long)r0 * lda;
        C += (long)r0 * sCm;
        if (EPI_GRAD) { ge.Y += (long)r0 * sCm; ge.sin_p += r0; ge.cos_p += r0; }
    }
    // K chunks of 16, 3 stages
    constexpr int KC = 16, STG = 3, PA = KC + 4;
    constexpr int PG_PB = NC + 4, PG_PC = NC + 2, NG = NC / 16, HC = NC / 2;
    const int stageA = Mpad * PA, stageB = KC * PG_PB;
    double *As = sm, *Bs = sm + STG * stageA;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int mg = warp / NG, ng = warp % NG;
    const int c0 = bx * NC;
    const double *Bb = B + (long)by * sBb + c0;
    double *Cb = C + (long)by * sCb + c0;
    const int nchunks = (K + KC - 1) / KC;
    const int colsleft = ncols - c0;                    // > 0, even

    // loaders: per-thread pointers set up once per chunk and advanced by constants (the loader's instruction count is comparable
    // to the tensor loop's at these short K); rows >= K and columns >= ncols are zero-filled through cp.async's ignore-src
    const int hA = tid & (KC / 2 - 1), rA0 = tid / (KC / 2), rAstep = blockDim.x / (KC / 2);
    const int hB = tid % HC, rB0 = tid / HC, rBstep = blockDim.x / HC;
    const bool coldead = 2 * hB >= colsleft;
    const long gAstep = (long)rAstep * lda, gBstep = (long)rBstep * sBk;
    auto load_chunk = [&](int kc, int st) {
        // A chunk: Mpad rows x 16 doubles (8 x 16 B per row); rows and K are zero padded in global memory
        double *as = As + st * stageA + rA0 * PA + 2 * hA;
        const double *ga = A + (long)rA0 * lda + kc * KC + 2 * hA;
#pragma unroll 1
        for (int r = rA0; r < Mpad; r += rAstep, as += rAstep * PA, ga += gAstep) cp_async16(as, ga);
        // B chunk: 16 rows x NC columns
        double *bs = Bs + st * stageB + rB0 * PG_PB + 2 * hB;
        const double *gb = Bb + (long)(kc * KC + rB0) * sBk + 2 * hB;
#pragma unroll 1
        for (int r = rB0; r < KC; r += rBstep, bs += rBstep * PG_PB, gb += gBstep)
            cp_async16_ign(bs, gb, coldead || kc * KC + r >= K);
    };

    // EPI_GRAD: 1/(r sin th) of the column pair this thread walks in phase 2 of the epilogue (q % HC = tid % HC because HC divides
    // the block size), loaded now so that the epilogue does not start with a global-load round trip
    double2 fcol = make_double2(0.0, 0.0);
    if (EPI_GRAD) {
        const int c = c0 + 2 * (tid % HC);                          // flat (k, i) column: c = k + Nr i
        if (c < ncols) { const int i = c / ge.Nr, k = c - i * ge.Nr; fcol.x = __ldg(ge.inv_r + k) * __ldg(ge.inv_sin_t + i); }
        if (c + 1 < ncols) { const int i = (c + 1) / ge.Nr, k = c + 1 - i * ge.Nr; fcol.y = __ldg(ge.inv_r + k) * __ldg(ge.inv_sin_t + i); }
    }
    double acc[MT][2][2];
#pragma unroll
    for (int a = 0; a < MT; a++)
#pragma unroll
        for (int b = 0; b < 2; b++) acc[a][b][0] = acc[a][b][1] = 0.0;

#pragma unroll
    for (int s = 0; s < STG - 1; s++) {
        if (s < nchunks) load_chunk(s, s);
        cp_async_commit();
    }
    for (int kc = 0; kc < nchunks; kc++) {
        cp_async_wait<STG - 2>();
        __syncthreads();
        if (kc + STG - 1 < nchunks) load_chunk(kc + STG - 1, (kc + STG - 1) % STG);
        cp_async_commit();
        const double *as = As + (kc % STG) * stageA + (mg * MT * 8 + g) * PA + t;
        const double *bs = Bs + (kc % STG) * stageB + t * PG_PB + ng * 16 + g;
        const int nks = min(KC / 4, (K - kc * KC + 3) >> 2);      // the last chunk may be short
#pragma unroll 4
        for (int ks = 0; ks < nks; ks++) {
            double af[MT], bf[2];
#pragma unroll
            for (int a = 0; a < MT; a++) af[a] = as[a * 8 * PA + ks * 4];
            bf[0] = bs[ks * 4 * PG_PB];
            bf[1] = bs[ks * 4 * PG_PB + 8];
#pragma unroll
            for (int a = 0; a < MT; a++) {
                dmma(acc[a][0][0], acc[a][0][1], af[a], bf[0]);
                dmma(acc[a][1][0], acc[a][1][1], af[a], bf[1]);
            }
        }
    }
    if (!EPI_GRAD) {
#pragma unroll
        for (int a = 0; a < MT; a++) {
            const int row = (mg * MT + a) * 8 + g;
            if (row >= M) continue;
#pragma unroll
            for (int b = 0; b < 2; b++) {
                const int col = ng * 16 + b * 8 + 2 * t;
                if (col < colsleft) *reinterpret_cast<double2 *>(Cb + (long)row * sCm + col) = make_double2(acc[a][b][0], acc[a][b][1]);
            }
        }
    } else {
        // two phases.  (1) every lane parks its accumulators (d_phi u) in shared memory (the pipeline buffers are free now) as an
        // [M][NC] tile.  (2) all threads walk the tile row-contiguously: c = d_phi u /(r sin th) with the thread's column factors,
        // coalesced 16-byte loads of W, coalesced stores of d_x and d_y, several independent loads in flight per thread.
        cp_async_wait<0>();
        __syncthreads();
        double *cs = sm;
        double *Yb = ge.Y + (long)by * ge.sYb + c0;
#pragma unroll
        for (int a = 0; a < MT; a++) {
            const int row = (mg * MT + a) * 8 + g;                       // longitude j
            if (row >= M) continue;
#pragma unroll
            for (int b = 0; b < 2; b++)
                *reinterpret_cast<double2 *>(cs + row * PG_PC + ng * 16 + b * 8 + 2 * t) = make_double2(acc[a][b][0], acc[a][b][1]);
        }
        __syncthreads();
        const int npair = min(NC, colsleft) >> 1;
        constexpr int UNR = 4;
        for (int q0 = tid; q0 < M * HC; q0 += UNR * blockDim.x) {
            double2 w[UNR];
            int row[UNR], cp2[UNR];
            bool ok[UNR];
#pragma unroll
            for (int z = 0; z < UNR; z++) {
                const int q = q0 + z * blockDim.x;
                row[z] = q / HC; cp2[z] = q % HC;
                ok[z] = q < M * HC && cp2[z] < npair;
                if (ok[z]) w[z] = *reinterpret_cast<const double2 *>(Cb + (long)row[z] * sCm + 2 * cp2[z]);
            }
#pragma unroll
            for (int z = 0; z < UNR; z++) {
                if (!ok[z]) continue;
                double2 c = *reinterpret_cast<const double2 *>(cs + row[z] * PG_PC + 2 * cp2[z]);
                c.x *= fcol.x; c.y *= fcol.y;
                const double sp = __ldg(ge.sin_p + row[z]), cp = __ldg(ge.cos_p + row[z]);
                *reinterpret_cast<double2 *>(Cb + (long)row[z] * sCm + 2 * cp2[z]) = make_double2(cp * w[z].x - sp * c.x, cp * w[z].y - sp * c.y);
                *reinterpret_cast<double2 *>(Yb + (long)row[z] * sCm + 2 * cp2[z]) = make_double2(sp * w[z].x + cp * c.x, sp * w[z].y + cp * c.y);
            }
        }
    }
}

// tiling of the row dimension chosen at build time: MT in {4,5,6} m-tiles per warp, mgroups warps along M
struct PhiTiling { int MT, mgroups, Mpad; };
static inline PhiTiling phi_tiling(int M) {
    const int mtiles = (M + 7) / 8;
    PhiTiling best = {6, (mtiles + 5) / 6, 0};
    int bestpad = best.mgroups * 6;
    for (int mt = 5; mt >= 4; mt--) {
        int gq = (mtiles + mt - 1) / mt;
        if (gq * mt < bestpad && gq <= 4) { best.MT = mt; best.mgroups = gq; bestpad = gq * mt; }
    }
    if (best.mgroups > 4) { best.MT = 6; best.mgroups = (mtiles + 5) / 6; }
    best.Mpad = best.mgroups * best.MT * 8;
    return best;
}
static inline size_t phi_smem_bytes(const PhiTiling &tl, int Mgrad = 0, int NC = PG_NCOL) {
    const int KC = 16, STG = 3, PA = KC + 4;
    const size_t pipe = (size_t)STG * ((size_t)tl.Mpad * PA + KC * (NC + 4)) * sizeof(double);
    const size_t tile = (size_t)Mgrad * (NC + 2) * sizeof(double);      // the gradient epilogue's tile reuses the pipeline buffers
    return pipe > tile ? pipe : tile;
}
// column tile width: 64, or 32 when 64-wide tiles would give fewer than 2 CTAs per SM (small states: more, smaller CTAs keep
// every SM busy and let several CTAs per SM overlap their load, product and store phases).  SP_PHI_NC overrides (experiments).
static inline int phi_ncol(int ncols, int nbatch, int num_sms) {
    static const int forced = [] { const char *e = getenv("SP_PHI_NC"); return e ? atoi(e) : 0; }();
    if (forced == 32 || forced == 64) return forced;
    const long ctas64 = (long)((ncols + 63) / 64) * nbatch;
    return ctas64 < 2L * num_sms ? 32 : 64;
}

// returns SP_ERR_UNSUPPORTED when the fast-path preconditions do not hold (caller falls back)
static sp_status launch_phi_gemm(const double *A, int lda, int M, const PhiTiling &tl, int K, const double *B, long sBk, long sBb,
                                 double *C, long sCm, long sCb, int ncols, int nbatch, cudaStream_t st, int num_sms,
                                 const PhiGradEpi *ge = nullptr) {
    if ((sBk | sBb | sCm | sCb | (long)ncols) & 1) return SP_ERR_UNSUPPORTED;
    if (((uintptr_t)B | (uintptr_t)C) & 15) return SP_ERR_UNSUPPORTED;
    if (tl.mgroups > 4) return SP_ERR_UNSUPPORTED;
    const int NC = phi_ncol(ncols, nbatch, num_sms);      // num_sms: SM count of the device the shell was built on
    // row blocks: products with two warp rows and many column tiles run as two CTAs of half the rows (measured: config 4
    // analysis -9 %, synthesis -4 %; config 3 d/dphi with the chain rule -7 %).  SP_PHI_MSPLIT overrides (experiments).
    static const int msplit_env = [] { const char *e = getenv("SP_PHI_MSPLIT"); return e ? atoi(e) : -1; }();
    const long ctas = (long)((ncols + NC - 1) / NC) * nbatch;
    int zs = (tl.mgroups == 2 && ctas >= 8L * num_sms) ? 2 : 1;
    if (msplit_env >= 1) zs = (tl.mgroups % msplit_env == 0) ? msplit_env : 1;
    PhiTiling tz = tl;
    tz.mgroups = tl.mgroups / zs; tz.Mpad = tl.Mpad / zs;
    // row blocks fastest in launch order when the operand they share is too large to wait in L2 (see the kernel)
    const int sfast = (zs > 1 && (double)K * ncols * nbatch * sizeof(double) > SP_SPLIT_FAST_BYTES) ? 1 : 0;
    const dim3 grid = sfast ? dim3(zs, (ncols + NC - 1) / NC, nbatch) : dim3((ncols + NC - 1) / NC, nbatch, zs);
    const dim3 block(tz.mgroups * (NC / 16) * 32);
#define SP_PG(MTV, EPIV, SM, GE)                                                                                              \
    if (NC == 32) k_phi_gemm<MTV, EPIV, 32><<<grid, block, SM, st>>>(A, lda, M, tl.Mpad, K, B, sBk, sBb, C, sCm, sCb, ncols, GE, sfast); \
    else k_phi_gemm<MTV, EPIV, 64><<<grid, block, SM, st>>>(A, lda, M, tl.Mpad, K, B, sBk, sBb, C, sCm, sCb, ncols, GE, sfast);
    if (ge) {
        if ((ge->sYb & 1) || ((uintptr_t)ge->Y & 15)) return SP_ERR_UNSUPPORTED;
        const size_t sm = phi_smem_bytes(tz, std::min(M, tz.Mpad), NC);
        if (sm > 227 * 1024) return SP_ERR_UNSUPPORTED;
        switch (tl.MT) {
            case 4: SP_PG(4, true, sm, *ge) break;
            case 5: SP_PG(5, true, sm, *ge) break;
            default: SP_PG(6, true, sm, *ge) break;
        }
        return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
    }
    const size_t sm = phi_smem_bytes(tz, 0, NC);
    PhiGradEpi none = {};
    switch (tl.MT) {
        case 4: SP_PG(4, false, sm, none) break;
        case 5: SP_PG(5, false, sm, none) break;
        default: SP_PG(6, false, sm, none) break;
    }
#undef SP_PG
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}
