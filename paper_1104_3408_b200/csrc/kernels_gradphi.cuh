// d/dphi of every field with the chain rule fused (eq. 17-19; 86-90 eq. 6), REFLECTION-FOLDED.
// FD_{Nphi} is an antisymmetric circulant, FD[j'][j] = g(j'-j), g(-d) = -g(d) (eq. 8).  With h = J/2 and, for jj = 0..h,
//     E_jj = (u_jj + u_{J-jj})/2,   O_jj = (u_jj - u_{J-jj})/2        (u_J = u_0; O_0 = O_h = 0)
//     Gp[j'][jj] = g(j'-jj) + g(j'+jj) (0 < jj < h), Gp[j'][0] = g(j'), Gp[j'][h] = g(j'-h);   Gm[j'][jj] = g(j'-jj) - g(j'+jj)
// the same sums regroup to
//     (d_phi u)[j'] = (Gm O)[j'] + (Gp E)[j'],      (d_phi u)[J-j'] = (Gm O)[j'] - (Gp E)[j'],      j' = 0..h,
// i.e. two (h+1) x (h+1) products instead of one J x J: half the DMMAs.
// CTA = NC (64, or 32 for small states: phi_ncol) columns of one field x all rows; K (= jj) in chunks of 8 through a 3-stage cp.async pipeline holding the rows
// u_jj and u_{J-jj} and the matching columns of Gm, Gp.  Warp (mg, ng) = MT row tiles x 2 column tiles, two accumulator
// sets (O and E products).  Epilogue: c = d_phi u /(r sin th); with W (written by k_grad_rtheta3 into the d_x slot)
//     d_x[j'] = cos(ph) W[j'] - sin(ph) c[j'],  d_y[j'] = sin(ph) W[j'] + cos(ph) c[j'],
// and the same for the mirrored row J-j' (cos(ph_{J-j'}) = cos(ph_j'), sin(ph_{J-j'}) = -sin(ph_j')).
#pragma once
#include "kernels_gemm2.cuh"

#define GF_KC 8
#define GF_STAGES 3
#define GF_PA 12

template <int MT, int NC>
__global__ void __launch_bounds__(NC * 8)
k_phi_grad_fold(const double *__restrict__ Gm, const double *__restrict__ Gp, int lda, int J, int Mpad,
                const double *__restrict__ U, long sUj, long sUb, double *__restrict__ X, double *__restrict__ Y, long sXb, int ncols,
                PhiGradEpi ge, int sfast) {
    extern __shared__ __align__(16) double sm[];
    constexpr int GF_PB = NC + 4, GF_PC = NC + 2, NG = NC / 16, HC = NC / 2;
    const int h = J >> 1, K = h + 1;
    int M = h + 1, r0 = 0;
    const int nzs = sfast ? gridDim.x : gridDim.z, bz = sfast ? blockIdx.x : blockIdx.z;      // grid orders as in k_phi_gemm
    const int bx = sfast ? blockIdx.y : blockIdx.x, by = sfast ? blockIdx.z : blockIdx.y;
    if (nzs > 1) {                                // row blocks: this CTA owns the rows j' in [r0, r0 + Mpad / gridDim.x) and their mirrors
        Mpad /= nzs;
        r0 = bz * Mpad;
        M = min(M - r0, Mpad);
        Gm += (long)r0 * lda;
        Gp += (long)r0 * lda;
    }
    const int stageA = 2 * Mpad * GF_PA, stageB = 2 * GF_KC * GF_PB;
    double *As = sm, *Bs = sm + GF_STAGES * stageA;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int mg = warp / NG, ng = warp % NG;
    const int c0 = bx * NC;
    const double *Ub = U + (long)by * sUb + c0;
    const int colsleft = ncols - c0;
    const int nchunks = (K + GF_KC - 1) / GF_KC;
    const int mtiles = (M + 7) >> 3;

    // loaders: per-thread pointers set up once per chunk and advanced by constants; dead rows / columns are zero-filled through
    // cp.async's ignore-src (see k_phi_gemm)
    const int hA = tid & 3, rA0 = tid >> 2, rAstep = blockDim.x >> 2;          // matrices: 4 x 16 B per row
    const int hB = tid % HC, rB0 = tid / HC, rBstep = blockDim.x / HC;         // field rows: NC/2 x 16 B per row
    const bool coldead = 2 * hB >= colsleft;
    const long gAstep = (long)rAstep * lda, gBstep = (long)rBstep * sUj;
    auto load_chunk = [&](int kc, int st) {
        double *as = As + st * stageA + rA0 * GF_PA + 2 * hA;
        const long ao = (long)rA0 * lda + kc * GF_KC + 2 * hA;
        const double *gm = Gm + ao, *gp = Gp + ao;
#pragma unroll 1
        for (int r = rA0; r < Mpad; r += rAstep, as += rAstep * GF_PA, gm += gAstep, gp += gAstep) {
            cp_async16(as, gm);
            cp_async16(as + Mpad * GF_PA, gp);
        }
        // rows jj (ascending) and their mirrors J - jj (descending; J -> 0)
        double *bs = Bs + st * stageB + rB0 * GF_PB + 2 * hB;
        const int jj0 = kc * GF_KC + rB0;
        const double *gu = Ub + (long)jj0 * sUj + 2 * hB, *gv = Ub + (long)(J - jj0) * sUj + 2 * hB;
#pragma unroll 1
        for (int r = rB0; r < GF_KC; r += rBstep, bs += rBstep * GF_PB, gu += gBstep, gv -= gBstep) {
            const int jj = kc * GF_KC + r;
            const bool dead = coldead || jj >= K;
            cp_async16_ign(bs, gu, dead);
            cp_async16_ign(bs + GF_KC * GF_PB, jj == 0 ? gu : gv, dead);
        }
    };

    // 1/(r sin th) of the column pair this thread walks in phase 2 of the epilogue (q % HC = tid % HC because HC divides the
    // block size), loaded now so that the epilogue does not start with a global-load round trip
    double2 fcol = make_double2(0.0, 0.0);
    {
        const int c = c0 + 2 * (tid % HC);                              // flat (k, i) column: c = k + Nr i
        if (c < ncols) { const int i = c / ge.Nr, k = c - i * ge.Nr; fcol.x = __ldg(ge.inv_r + k) * __ldg(ge.inv_sin_t + i); }
        if (c + 1 < ncols) { const int i = (c + 1) / ge.Nr, k = c + 1 - i * ge.Nr; fcol.y = __ldg(ge.inv_r + k) * __ldg(ge.inv_sin_t + i); }
    }
    double aO[MT][2][2], aE[MT][2][2];
#pragma unroll
    for (int a = 0; a < MT; a++)
#pragma unroll
        for (int b = 0; b < 2; b++) aO[a][b][0] = aO[a][b][1] = aE[a][b][0] = aE[a][b][1] = 0.0;

#pragma unroll
    for (int s = 0; s < GF_STAGES - 1; s++) {
        if (s < nchunks) load_chunk(s, s);
        cp_async_commit();
    }
    for (int kc = 0; kc < nchunks; kc++) {
        cp_async_wait<GF_STAGES - 2>();
        __syncthreads();
        if (kc + GF_STAGES - 1 < nchunks) load_chunk(kc + GF_STAGES - 1, (kc + GF_STAGES - 1) % GF_STAGES);
        cp_async_commit();
        const double *as = As + (kc % GF_STAGES) * stageA + (mg * MT * 8 + g) * GF_PA + t;
        const double *bs = Bs + (kc % GF_STAGES) * stageB + t * GF_PB + ng * 16 + g;
#pragma unroll
        for (int ks = 0; ks < GF_KC / 4; ks++) {
            double bE[2], bO[2];
#pragma unroll
            for (int b = 0; b < 2; b++) {
                const double x = bs[ks * 4 * GF_PB + b * 8], y = bs[(GF_KC + ks * 4) * GF_PB + b * 8];
                bE[b] = 0.5 * (x + y); bO[b] = 0.5 * (x - y);
            }
#pragma unroll
            for (int a = 0; a < MT; a++) {
                if ((mg * MT + a) < mtiles) {                               // warp-uniform: skip dead row tiles
                    const double am = as[a * 8 * GF_PA + ks * 4], ap = as[(Mpad + a * 8) * GF_PA + ks * 4];
#pragma unroll
                    for (int b = 0; b < 2; b++) {
                        dmma(aO[a][b][0], aO[a][b][1], am, bO[b]);
                        dmma(aE[a][b][0], aE[a][b][1], ap, bE[b]);
                    }
                }
            }
        }
    }
    // ---- epilogue, two phases.  (1) every lane unfolds its accumulators to d_phi u and parks them in shared memory (the pipeline
    // buffers are free now) as a [J][64] tile.  (2) all threads walk the tile row-contiguously: c = d_phi u /(r sin th) with the
    // thread's column factors, coalesced 16-byte loads of W, coalesced stores of d_x and d_y, many independent loads in flight.
    cp_async_wait<0>();
    __syncthreads();
    double *cs = sm;                                                        // [2 Mpad][GF_PC]: rows j', then their mirrors J - j'
#pragma unroll
    for (int a = 0; a < MT; a++) {
        const int row = (mg * MT + a) * 8 + g;                          // local row; j' = r0 + row in [0, h]
        if (row >= M) continue;
        const bool mirrored = r0 + row > 0 && r0 + row < h;
#pragma unroll
        for (int b = 0; b < 2; b++) {
            const int col = ng * 16 + b * 8 + 2 * t;
            *reinterpret_cast<double2 *>(cs + row * GF_PC + col) = make_double2(aO[a][b][0] + aE[a][b][0], aO[a][b][1] + aE[a][b][1]);
            if (mirrored)
                *reinterpret_cast<double2 *>(cs + (Mpad + row) * GF_PC + col) =
                    make_double2(aO[a][b][0] - aE[a][b][0], aO[a][b][1] - aE[a][b][1]);
        }
    }
    __syncthreads();
    double *Xb = X + (long)by * sXb + c0, *Yb = Y + (long)by * sXb + c0;
    const int npair = min(NC, colsleft) >> 1;                          // column pairs of this tile
    constexpr int UNR = 4;
    for (int q0 = tid; q0 < 2 * Mpad * HC; q0 += UNR * blockDim.x) {
        double2 w[UNR];
        int lrow[UNR], row[UNR], cp2[UNR];
        bool ok[UNR];
#pragma unroll
        for (int z = 0; z < UNR; z++) {
            const int q = q0 + z * blockDim.x;
            lrow[z] = q / HC; cp2[z] = q % HC;
            const bool mir = lrow[z] >= Mpad;
            const int lr = lrow[z] - (mir ? Mpad : 0), jp = r0 + lr;         // j' of this tile row
            row[z] = mir ? J - jp : jp;                                      // longitude j
            ok[z] = q < 2 * Mpad * HC && lr < M && cp2[z] < npair && (!mir || (jp > 0 && jp < h));
            if (ok[z]) w[z] = *reinterpret_cast<const double2 *>(Xb + (long)row[z] * sUj + 2 * cp2[z]);
        }
#pragma unroll
        for (int z = 0; z < UNR; z++) {
            if (!ok[z]) continue;
            double2 c = *reinterpret_cast<const double2 *>(cs + lrow[z] * GF_PC + 2 * cp2[z]);
            c.x *= fcol.x; c.y *= fcol.y;
            const double sp = __ldg(ge.sin_p + row[z]), cp = __ldg(ge.cos_p + row[z]);
            *reinterpret_cast<double2 *>(Xb + (long)row[z] * sUj + 2 * cp2[z]) = make_double2(cp * w[z].x - sp * c.x, cp * w[z].y - sp * c.y);
            *reinterpret_cast<double2 *>(Yb + (long)row[z] * sUj + 2 * cp2[z]) = make_double2(sp * w[z].x + cp * c.x, sp * w[z].y + cp * c.y);
        }
    }
}

static inline size_t gradfold_smem_bytes(int Mpad, int J, int NC = PG_NCOL) {      // Mpad = rows per CTA
    (void)J;
    const size_t pipe = (size_t)GF_STAGES * ((size_t)2 * Mpad * GF_PA + 2 * GF_KC * (NC + 4)) * sizeof(double);
    const size_t tile = (size_t)2 * Mpad * (NC + 2) * sizeof(double);                 // the epilogue tile reuses the pipeline buffers
    return pipe > tile ? pipe : tile;
}
