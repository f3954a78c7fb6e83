// Fused stages of the Yn tensor filter (eq. 51-56, 33, 31, 60; the paper names running these products together
// as its next optimisation):
//
//   k_fan   F1 + F2: dyad projection (eq. 54-56) + phi-reflection fold + phi analysis (eq. 33) in ONE kernel.  A CTA owns NC
//           consecutive (k, i) columns of ONE tensor, for all longitudes and all components: the raw Cartesian components are
//           staged once in shared memory [component][j][column], projected and folded IN PLACE (a thread owns the points j and
//           J - j of a column, all components), and the folded tile is the B operand of the two Fourier products (cosine block
//           a_0..a_L over E rows, sine block b_1..b_L over O rows), whose matrices stream through a cp.async pipeline in K chunks.
//           The spin-weight components never exist in global memory.
//   k_fsyn  F4 + F5: phi synthesis (eq. 31) + unfold + recombination with the conjugate dyad (eq. 56, 60) in ONE kernel.  A CTA
//           owns NC columns of one tensor; the filtered coefficient rows of all components are staged once in shared memory; warp w
//           owns the longitudes jj = 8w..8w+7 and their mirrors J - jj for ALL components (one n-tile per component and column
//           block), so that after the two products (e_jj from the cosine rows, o_jj from the sine rows) a lane holds every
//           component of its grid points in registers: the unfold f_jj = e + o, f_{J-jj} = e - o and the inverse dyad
//           transformation are lane-local and the Cartesian components go straight to global memory.
//
// Both kernels are PERSISTENT: a CTA walks the work items (tensor of the launch group, column tile) with stride gridDim.x and
// stages the next item's tile with cp.async into a second buffer while the current one is projected and multiplied, so the HBM
// reads of one item run under the tensor work of the previous one (with one buffer the grid equals the item count).
// Both kernels keep the data tile resident in shared memory (it is read from HBM exactly once) and take the A fragments of the
// small Fourier matrices straight from global memory (read-only path: the matrices are shared by every CTA and stay in L1/L2), so
// the products run without any block-level synchronisation.  Shared-memory layout of the data tiles: pitch NC with an XOR swizzle
// of the column by the row (no padding), so that the DMMA B-fragment loads (4 rows x 8 columns per warp) and the pointwise
// phase are both conflict free.
#pragma once
#include "kernels_filter.cuh"
#include "kernels_gemm2.cuh"

struct FusedParams {
    int Nr, Nt, L, vec, MC;              // J = 2 Nt; vec = Nr * Nt columns per longitude; MC = 2L + 1 coefficient rows per dof
    long npts, dofsz;                    // field stride; coefficient array stride per dof (MC4 * vec)
    const double *sin_t, *cos_t, *sin_p, *cos_p;
    const double *Ac, *As;               // analysis: [Mp][ldc] rows a_0..a_L over jj = 0..h; [Mp][lds] rows b_1..b_L over q, jj = h-1-q
    int Mp, ldc, lds;
    const double *Sc, *Ss;               // synthesis: [Jp][ldk] rows jj = 0..h over m = 0..L; [Jp][ldk] rows jj (0 and h zero) over b_1..b_L
    int Jp, ldk;
    int WM, WN;                          // k_fan: warps along the coefficient rows / along the columns (further warps only stage and project)
    int ngroup, nbuf, zs;                // tensors in this launch; tile buffers (1 or 2); k_fsyn: CTAs sharing the longitudes of a column tile
};

// XOR swizzle of the column index by the row of a data tile of pitch NC (NC = 4: rows of 32 bytes need none)
template <int NC> __device__ __forceinline__ int fu_sw(int row) { return NC >= 16 ? ((row & 3) << 2) : NC == 8 ? ((row & 2) << 1) : 0; }

// N dimension of the products: n = component * NC + column; an n-tile is 8 consecutive n (NC = 4: two components x 4 columns)
template <int TT, int NC, int MT, int NTW, int MAXT>
__global__ void __launch_bounds__(MAXT)
k_fan(const __grid_constant__ TensorArgsGroup tg, const __grid_constant__ FusedParams p, const double *__restrict__ src,
      double *__restrict__ coef) {
    constexpr int nc = TTInfo<TT>::nc, NTOT = nc * NC, PPR = NC / 2;
    static_assert(NTOT % 8 == 0, "components x columns must fill whole n-tiles");
    extern __shared__ __align__(16) double sm[];          // nbuf x (data tile [nc][J][NC] + 4 zero rows)
    const int J = 2 * p.Nt, h = p.Nt, CS = J * NC, XSZ = nc * CS + 4 * NC;
    const int tid = threadIdx.x, nthr = blockDim.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int WM = p.WM, wm = warp % WM, wn = warp / WM;
    const bool mma_warp = wn < p.WN;
    const int ntx = (p.vec + NC - 1) / NC, nitems = ntx * p.ngroup;

    // stage the raw components of an item: [component][j][NC columns], 16-byte pieces, dead columns zero-filled
    auto stage = [&](int item, int XB) {
        const TensorArgs &ta = tg.t[item / ntx];
        const int c0 = (item % ntx) * NC, colsleft = p.vec - c0;
        for (int q = tid; q < J * PPR; q += nthr) {
            const int row = q / PPR, cp2 = 2 * (q % PPR);
            const bool dead = cp2 >= colsleft;
            const double *gsrc = src + (size_t)row * p.vec + c0 + (dead ? 0 : cp2);
            const int xo = XB + row * NC + (cp2 ^ fu_sw<NC>(row));
#pragma unroll
            for (int c = 0; c < nc; c++) cp_async16_ign(&sm[xo + c * CS], gsrc + (size_t)ta.field[c] * p.npts, dead);
        }
        cp_async_commit();
    };
    for (int q = tid; q < p.nbuf * 4 * NC; q += nthr) sm[(q / (4 * NC)) * XSZ + nc * CS + q % (4 * NC)] = 0.0;
    int item = blockIdx.x;
    if (item >= nitems) return;
    stage(item, 0);
    // B fragment of lane (g, t) in n-tile nt: n = 8 nt + g  ->  (component, column); pre[b] = component * CS + column
    int pre[NTW];
#pragma unroll
    for (int b = 0; b < NTW; b++) {
        const int n = min((wn * NTW + b) * 8 + g, NTOT - 1);
        pre[b] = (n / NC) * CS + (n % NC);
    }
    const int mtiles = p.Mp >> 3, npass = (mtiles + WM * MT - 1) / (WM * MT);

    for (int itn = 0; item < nitems; item += gridDim.x, itn++) {
        const int XB = (p.nbuf > 1 ? (itn & 1) : 0) * XSZ;
        const TensorArgs &ta = tg.t[item / ntx];
        const int c0 = (item % ntx) * NC, colsleft = p.vec - c0;
        cp_async_wait<0>();
        __syncthreads();              // this item's tile has landed; every warp is done with the products of the previous item
        if (p.nbuf > 1 && item + gridDim.x < nitems) stage(item + gridDim.x, XSZ - XB);

        // ---- F1: project and fold in place.  One work unit = the grid points (jj, column) and (J - jj, column), all components.
        for (int it = tid; it < (h + 1) * NC; it += nthr) {
            const int jj = it / NC, col = it % NC;
            if (col >= colsleft) continue;
            const int i = (c0 + col) / p.Nr;
            const double st = __ldg(p.sin_t + i), ct = __ldg(p.cos_t + i);
            const int r2 = J - jj;
            const bool paired = (jj != 0) && (jj != h);
            const int o1 = XB + jj * NC + (col ^ fu_sw<NC>(jj)), o2 = XB + r2 * NC + (col ^ fu_sw<NC>(r2));
            const double sp = __ldg(p.sin_p + jj), cp = __ldg(p.cos_p + jj);
            double in[nc], a[nc], b[nc];
#pragma unroll
            for (int c = 0; c < nc; c++) in[c] = sm[o1 + c * CS];
            const Trig t1 = {st, ct, sp, cp};
            tensor_transform<TT, false>(t1, in, a);
            if (paired) {
#pragma unroll
                for (int c = 0; c < nc; c++) in[c] = sm[o2 + c * CS];
                const Trig t2 = {st, ct, -sp, cp};            // phi_{J-jj} = 2 pi - phi_jj
                tensor_transform<TT, false>(t2, in, b);
#pragma unroll
                for (int c = 0; c < nc; c++) { sm[o1 + c * CS] = a[c] + b[c]; sm[o2 + c * CS] = a[c] - b[c]; }
            } else {
#pragma unroll
                for (int c = 0; c < nc; c++) sm[o1 + c * CS] = a[c];
            }
        }
        __syncthreads();
        if (!mma_warp) continue;                              // the further warps only stage and project

        // ---- F2: the two Fourier products on the folded tile (A fragments from global memory)
        for (int blk = 0; blk < 2; blk++) {
            const int K = blk ? ((p.L > 0) ? h - 1 : 0) : h + 1, M = blk ? p.L : p.L + 1, brow0 = blk ? h + 1 : 0;
            const double *A = blk ? p.As : p.Ac;
            const int lda = blk ? p.lds : p.ldc, nks = (K + 3) >> 2;
            if (K <= 0) continue;
            for (int pm = 0; pm < npass; pm++) {
                const int row0 = (pm * WM + wm) * MT * 8 + g;                 // this lane's rows: row0 + 8 a
                const double *ap[MT];
#pragma unroll
                for (int a = 0; a < MT; a++) ap[a] = A + (size_t)min(row0 + 8 * a, p.Mp - 1) * lda + t;
                double acc[MT][NTW][2];
#pragma unroll
                for (int a = 0; a < MT; a++)
#pragma unroll
                    for (int b = 0; b < NTW; b++) acc[a][b][0] = acc[a][b][1] = 0.0;
                // small warp tiles are latency bound (one read-only load per few DMMAs): unroll deeper so that the fragment loads of
                // several k-steps are in flight
#pragma unroll(MT * NTW <= 6 ? 8 : MT * NTW <= 9 ? 4 : 2)
                for (int ks = 0; ks < nks; ks++) {
                    const int krow = brow0 + ks * 4 + t;
                    const int ro = XB + krow * NC, swz = fu_sw<NC>(krow);
                    double af[MT], bf[NTW];
#pragma unroll
                    for (int a = 0; a < MT; a++) af[a] = __ldg(ap[a] + ks * 4);
#pragma unroll
                    for (int b = 0; b < NTW; b++) bf[b] = sm[(pre[b] ^ swz) + ro];
#pragma unroll
                    for (int a = 0; a < MT; a++)
#pragma unroll
                        for (int b = 0; b < NTW; b++) dmma(acc[a][b][0], acc[a][b][1], af[a], bf[b]);
                }
                // epilogue of this (block, row pass): coefficient rows mc = m (cosine block), L + m (sine block, m = row + 1)
#pragma unroll
                for (int b = 0; b < NTW; b++) {
                    const int n = (wn * NTW + b) * 8 + 2 * t, comp = n / NC, col = n % NC;
                    if (n >= NTOT || col >= colsleft) continue;
                    double *dst = coef + (size_t)(ta.dof0 + comp) * p.dofsz + c0 + col;
#pragma unroll
                    for (int a = 0; a < MT; a++) {
                        const int row = row0 + 8 * a;
                        if (row >= M) continue;
                        const int mc = blk ? p.L + 1 + row : row;
                        *reinterpret_cast<double2 *>(dst + (size_t)mc * p.vec) = make_double2(acc[a][b][0], acc[a][b][1]);
                    }
                }
            }
        }
    }
}

template <int NC> static inline size_t fan_smem_bytes(int nc, int J, int nbuf) { return (size_t)nbuf * ((size_t)nc * J * NC + 4 * NC) * sizeof(double); }


// ---------------------------------------------------------------------------------------------------------------------
template <int TT, int CBW>
__global__ void __launch_bounds__(256)
k_fsyn(const __grid_constant__ TensorArgsGroup tg, const __grid_constant__ FusedParams p, const double *__restrict__ coef,
       double *__restrict__ dst) {
    constexpr int nc = TTInfo<TT>::nc, NC = 8 * CBW, PPR = NC / 2;
    extern __shared__ __align__(16) double sm[];          // nbuf x (coefficient tile [nc][MC][NC] + 4 zero rows)
    const int J = 2 * p.Nt, h = p.Nt, MC = p.MC, L = p.L, CS = MC * NC, XSZ = nc * CS + 4 * NC;
    const int tid = threadIdx.x, nthr = blockDim.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    // work item = (tensor, column tile, longitude block): zs CTAs share a column tile, each owns 8 longitudes per warp
    const int ntx = (p.vec + NC - 1) / NC, nitems = ntx * p.zs * p.ngroup;

    auto stage = [&](int item, int XB) {
        const TensorArgs &ta = tg.t[item / (ntx * p.zs)];
        const int c0 = ((item / p.zs) % ntx) * NC, colsleft = p.vec - c0;
        for (int q = tid; q < MC * PPR; q += nthr) {
            const int row = q / PPR, cp2 = 2 * (q % PPR);
            const bool dead = cp2 >= colsleft;
            const double *gsrc = coef + (size_t)ta.dof0 * p.dofsz + (size_t)row * p.vec + c0 + (dead ? 0 : cp2);
            const int co = XB + row * NC + (cp2 ^ fu_sw<NC>(row));
#pragma unroll
            for (int c = 0; c < nc; c++) cp_async16_ign(&sm[co + c * CS], gsrc + (size_t)c * p.dofsz, dead);
        }
        cp_async_commit();
    };
    for (int q = tid; q < p.nbuf * 4 * NC; q += nthr) sm[(q / (4 * NC)) * XSZ + nc * CS + q % (4 * NC)] = 0.0;
    int item = blockIdx.x;
    if (item >= nitems) return;
    stage(item, 0);
    const int nks = (L + 4) >> 2;                         // k-steps over m = 0..L; Ss is zero beyond its L columns

    for (int itn = 0; item < nitems; item += gridDim.x, itn++) {
        const int XB = (p.nbuf > 1 ? (itn & 1) : 0) * XSZ;
        const TensorArgs &ta = tg.t[item / (ntx * p.zs)];
        const int c0 = ((item / p.zs) % ntx) * NC, colsleft = p.vec - c0;
        const int jj = ((item % p.zs) * (nthr >> 5) + warp) * 8 + g;          // this lane's longitude (and its mirror J - jj)
        cp_async_wait<0>();
        __syncthreads();              // this item's tile has landed; every warp is done with the previous item
        if (p.nbuf > 1 && item + gridDim.x < nitems) stage(item + gridDim.x, XSZ - XB);
        if (jj - g > h) continue;                             // a warp beyond the last longitude tile
        // ---- F4: e_jj = sum_m Sc[jj][m] a~_m (rows mc = m), o_jj = sum_m Ss[jj][m-1] b~_m (rows mc = L + m)
        const double *scp = p.Sc + (size_t)min(jj, p.Jp - 1) * p.ldk + t, *ssp = p.Ss + (size_t)min(jj, p.Jp - 1) * p.ldk + t;
        double accE[nc][CBW][2], accO[nc][CBW][2];
#pragma unroll
        for (int c = 0; c < nc; c++)
#pragma unroll
            for (int b = 0; b < CBW; b++) accE[c][b][0] = accE[c][b][1] = accO[c][b][0] = accO[c][b][1] = 0.0;
#pragma unroll(nc * CBW <= 4 ? 8 : nc * CBW <= 8 ? 4 : 2)
        for (int ks = 0; ks < nks; ks++) {
            const int kr = ks * 4 + t, krs = L + 1 + kr;
            const double ac = __ldg(scp + ks * 4), asn = __ldg(ssp + ks * 4);
            const int co = XB + kr * NC, so = XB + krs * NC, swz = fu_sw<NC>(kr), sws = fu_sw<NC>(krs);
#pragma unroll
            for (int c = 0; c < nc; c++)
#pragma unroll
                for (int b = 0; b < CBW; b++) {
                    dmma(accE[c][b][0], accE[c][b][1], ac, sm[c * CS + co + ((b * 8 + g) ^ swz)]);
                    dmma(accO[c][b][0], accO[c][b][1], asn, sm[c * CS + so + ((b * 8 + g) ^ sws)]);
                }
        }
        // ---- F5: unfold and recombine, lane-local.  Lane (g, t) holds e_jj and o_jj of every component at the columns cb*8 + 2t, +1.
        if (jj > h) continue;
        const bool paired = (jj != 0) && (jj != h);
        const int r2 = J - jj;
        const double sp1 = __ldg(p.sin_p + jj), cp1 = __ldg(p.cos_p + jj);
#pragma unroll
        for (int b = 0; b < CBW; b++)
#pragma unroll
            for (int x = 0; x < 2; x++) {
                const int col = b * 8 + 2 * t + x;
                if (col >= colsleft) continue;
                const int i = (c0 + col) / p.Nr;
                const double st = __ldg(p.sin_t + i), ct = __ldg(p.cos_t + i);
                double a[nc], out[nc];
#pragma unroll
                for (int c = 0; c < nc; c++) a[c] = accE[c][b][x] + accO[c][b][x];
                const Trig t1 = {st, ct, sp1, cp1};
                tensor_transform<TT, true>(t1, a, out);
                double *d1 = dst + (size_t)jj * p.vec + c0 + col;
#pragma unroll
                for (int c = 0; c < nc; c++) d1[(size_t)ta.field[c] * p.npts] = out[c];
                if (paired) {
#pragma unroll
                    for (int c = 0; c < nc; c++) a[c] = accE[c][b][x] - accO[c][b][x];
                    const Trig t2 = {st, ct, -sp1, cp1};          // phi_{J-jj} = 2 pi - phi_jj
                    tensor_transform<TT, true>(t2, a, out);
                    double *d2 = dst + (size_t)r2 * p.vec + c0 + col;
#pragma unroll
                    for (int c = 0; c < nc; c++) d2[(size_t)ta.field[c] * p.npts] = out[c];
                }
            }
    }
}

static inline size_t fsyn_smem_bytes(int nc, int MC, int NC, int nbuf) { return (size_t)nbuf * ((size_t)nc * MC * NC + 4 * NC) * sizeof(double); }
