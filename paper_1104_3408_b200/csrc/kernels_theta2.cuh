// theta step of the Yn filter (eq. 61-62; 374-376), shared-memory staged.
//   coef[dof][mc][i][k]  (mc = m: a_m, m = 0..L; mc = L+m: b_m, m = 1..L)  ->  cout, same layout
// CTA = (component, m, block of 36 radii).  K (= latitude ii) is walked in chunks of 16 through a 3-stage
// cp.async pipeline holding the F^n_m rows (and F^{-n}_m for complex components) and the raw coefficient
// rows a_m, b_m (real) or a^r, b^r, a^i, b^i (complex) of the CTA's radii.
// Warp (mg, ng): MT latitude tiles x NT column tiles; a column tile is 4 radii x {v = 0, 1} interleaved
// (col = 2k + v), so a lane's accumulator pair is the (v=0, v=1) pair of one radius:
//   real (n = 0):  v=0: a~_m = F^0_m a_m,  v=1: b~_m = F^0_m b_m
//   complex spin n, m > 0 (reading Q12, F^n_{-m} = F^{-n}_m by eq. 47):
//       (p, q) = F^n_m    [(a^r + b^i)/2 , (a^i - b^r)/2]      = (Re, Im) c~_{+m}
//       (s, t) = F^{-n}_m [(a^r - b^i)/2 , (a^i + b^r)/2]      = (Re, Im) c~_{-m}
//       a~^r = p + s, b~^r = t - q, a~^i = q + t, b~^i = p - s
//   complex, m = 0:  a~^r_0 = F^n_0 a^r_0, a~^i_0 = F^n_0 a^i_0.
#pragma once
#include "kernels_gemm2.cuh"

#define TH_RC 36                        // radii per CTA = 9 column tiles = NT tiles per warp x (9 / NT) warp columns
// coefficient tile in shared memory, two layouts (measured): NT = 1 (many narrow warps): row pitch 38 (rows t = 0..3 land 6
// eight-byte slots apart mod 16) and array pitch = 8 mod 16 with the arrays a lane pair (v = 0, 1) reads together as neighbours:
// conflict-free fragments (config 4: 0.94 -> 0.89 ms); NT = 3: row pitch 37, arrays back to back (config 3: 61 us against 63.5)
#define TH_PKB_OF(NT) ((NT) == 1 ? 38 : 37)
#define TH_ARR_OF(NT) (TH_KC * TH_PKB_OF(NT) + ((NT) == 1 ? 8 : 0))
#define TH_KC 16
#define TH_STAGES 3
#define TH_PA 20

__device__ __forceinline__ void cp_async8(void *smem, const void *gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gmem));
}

// 8-byte cp.async; with ignore = true the source is not read and zeros are written
__device__ __forceinline__ void cp_async8_ign(void *smem, const void *gmem, bool ignore) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %2, 0;\n cp.async.ca.shared.global [%0], [%1], 8, p;\n}\n" ::"r"(s), "l"(gmem), "r"((int)ignore));
}

struct ThetaComp2 { int dof; int n; };
#define SP_THETA2_BATCH 96
struct ThetaBatch2 { ThetaComp2 c[SP_THETA2_BATCH]; };

// F2: [7][L+1][Nt8][Nt8] zero padded
// NT = column tiles per warp: 3 (3 warp columns, 72 accumulator registers for complex components) or 1 (9 warp columns,
// three times as many warps with a third of the registers).  Which one is faster depends on the grid; sp_build_matrices
// times both on the device and keeps the winner.
template <int MT, int NT, bool CPLX>
__global__ void __launch_bounds__(NT == 3 ? 384 : 896, 1)
k_theta2(ThetaBatch2 comps, const double *__restrict__ F2, int L, int Nt, int Nt8, int Nr, int MC4, int mgroups, int rsplit,
         const double *__restrict__ coef, double *__restrict__ cout, int sfast) {
    extern __shared__ __align__(16) double sm[];
    constexpr int NMAT = CPLX ? 2 : 1, NARR = CPLX ? 4 : 2;
    const ThetaComp2 cmp = comps.c[blockIdx.y];
    const int m = sfast ? blockIdx.x / rsplit : blockIdx.x;
    // sfast (large launches): blockIdx.x = m * rsplit + row block (the row blocks of one (component, m, radial block) read the same coefficient rows: neighbours in
    // launch order, so the second one finds them in L2), blockIdx.z = radial block; otherwise blockIdx.x = m, blockIdx.z = radial block * rsplit + row block: with rsplit = 2 a CTA owns half of the latitudes (rows of F^n_m), so its F tile
    // halves and two CTAs share an SM at large Ntheta; both row blocks read the same coefficient rows
    const int zr = sfast ? blockIdx.x % rsplit : blockIdx.z % rsplit, k0 = (sfast ? blockIdx.z : blockIdx.z / rsplit) * TH_RC;
    const int Nt8c = Nt8 / rsplit, r0 = zr * Nt8c;                  // rows of this CTA
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int mg = warp % mgroups, ng = warp / mgroups, nwarps = blockDim.x >> 5;
    const size_t vec = (size_t)Nt * Nr, dofsz = (size_t)MC4 * vec, fsz = (size_t)Nt8 * Nt8;
    const int mca = m;                                         // rows a_0..a_L, then b_1..b_L (b_m = row L + m: offset offAB below)
    constexpr int TH_PKB = TH_PKB_OF(NT), TH_ARR = TH_ARR_OF(NT);
    const int stageA = NMAT * Nt8c * TH_PA, stageB = NARR * TH_ARR;
    // shared-memory slot of source array arr: the pairs a lane pair (v = 0, 1) reads together are neighbours
    auto slot = [](int arr) { return CPLX ? ((arr == 0) ? 0 : (arr == 2) ? 1 : (arr == 3) ? 2 : 3) : arr; };
    // offset of (array, row) in a stage of the coefficient tile
    auto brow = [&](int arr, int r) { return NT == 1 ? slot(arr) * TH_ARR + r * TH_PKB : (arr * TH_KC + r) * TH_PKB; };
    // only min(TH_STAGES, K chunks) stages are allocated (theta2_smem_bytes): short K leaves room for more CTAs per SM
    double *As = sm, *Bs = sm + min(TH_STAGES, (Nt8 + TH_KC - 1) / TH_KC) * stageA;
    const int nrad = min(TH_RC, Nr - k0);
    // source arrays: real: [a_m, b_m]; complex: [a^r, b^r, a^i, b^i]
    const double *srcR = coef + (size_t)cmp.dof * dofsz + k0;            // arr = 2*part + (0: a_m, 1: b_m)
    const double *F0 = F2 + ((size_t)(3 + cmp.n) * (L + 1) + m) * fsz;
    const long dF = CPLX ? -2L * cmp.n * (long)(L + 1) * (long)fsz : 0L;   // F^{-n}_m relative to F^n_m
    const int nchunks = (Nt8 + TH_KC - 1) / TH_KC;

    // loaders.  Their instruction count matters (at 3 K-chunks per CTA they run as often as the tensor loop), so every address
    // is a pointer or shared-memory offset set up once per chunk and advanced by a constant; dead rows / columns are zero-filled
    // by cp.async with the ignore-src predicate (no divergent store path).
    const int hF = tid & 7, rF0 = tid >> 3, rFstep = blockDim.x >> 3;          // F tile: 8 sixteen-byte pieces per row
    const size_t offAB = (size_t)L * vec;                                       // b_m relative to a_m
    const double *srcA = srcR + (size_t)mca * vec + lane;                       // a_m rows of the (real part of the) component
    const bool live0 = lane < nrad, live1 = lane + 32 < nrad, lane_hi = lane < TH_RC - 32;
    auto load_chunk = [&](int kc, int st) {
        double *as = As + st * stageA + rF0 * TH_PA + 2 * hF;
        if (kc * TH_KC + 2 * hF < Nt8) {
            const double *fs = F0 + (r0 + rF0) * Nt8 + kc * TH_KC + 2 * hF;
            const int fstep = rFstep * Nt8;
#pragma unroll 1
            for (int r = rF0; r < Nt8c; r += rFstep, as += rFstep * TH_PA, fs += fstep) {
                cp_async16(as, fs);
                if (CPLX) cp_async16(as + Nt8c * TH_PA, fs + dF);
            }
        } else {
#pragma unroll 1
            for (int r = rF0; r < Nt8c; r += rFstep, as += rFstep * TH_PA) {
                as[0] = 0.0; as[1] = 0.0;
                if (CPLX) { as[Nt8c * TH_PA] = 0.0; as[Nt8c * TH_PA + 1] = 0.0; }
            }
        }
        // raw coefficient rows: one (array, latitude) row of 36 radii per warp iteration, lane = radius
        const int kbase = kc * TH_KC;
        const double *g0 = srcA + (size_t)(kbase + warp) * Nr;
        double *bs = Bs + st * stageB + lane;
        const int gstep = nwarps * Nr, sstep = nwarps * TH_PKB;
#pragma unroll
        for (int arr = 0; arr < NARR; arr++) {
            const double *gp = g0 + (arr >> 1) * dofsz + (arr & 1) * offAB;
            double *sp = bs + brow(arr, warp);
            const bool arrdead = (m == 0) && (arr & 1);                                 // b_0 does not exist
#pragma unroll 1
            for (int r = warp; r < TH_KC; r += nwarps, gp += gstep, sp += sstep) {
                const bool dead = arrdead || kbase + r >= Nt;
                cp_async8_ign(sp, gp, dead || !live0);
                if (lane_hi) cp_async8_ign(sp + 32, gp + 32, dead || !live1);
            }
        }
    };

    double acc[NMAT][MT][NT][2];
#pragma unroll
    for (int x = 0; x < NMAT; x++)
#pragma unroll
        for (int a = 0; a < MT; a++)
#pragma unroll
            for (int b = 0; b < NT; b++) acc[x][a][b][0] = acc[x][a][b][1] = 0.0;

#pragma unroll
    for (int s = 0; s < TH_STAGES - 1; s++) {
        if (s < nchunks) load_chunk(s, s);
        cp_async_commit();
    }
    const int v = g & 1, kq = g >> 1;
    // B-fragment sources of this lane: real: arr v; complex: X = v ? a^i : a^r, Y = v ? b^r : b^i (sign -1 if v)
    const int arrX = CPLX ? (v ? 2 : 0) : v, arrY = CPLX ? (v ? 1 : 3) : 0;
    const double ysgn = v ? -0.5 : 0.5, xscl = (m > 0) ? 0.5 : 1.0;
    for (int kc = 0; kc < nchunks; kc++) {
        cp_async_wait<TH_STAGES - 2>();
        __syncthreads();
        if (kc + TH_STAGES - 1 < nchunks) load_chunk(kc + TH_STAGES - 1, (kc + TH_STAGES - 1) % TH_STAGES);
        cp_async_commit();
        const double *as = As + (kc % TH_STAGES) * stageA + (mg * MT * 8 + g) * TH_PA + t;
        const double *bs = Bs + (kc % TH_STAGES) * stageB;
#pragma unroll
        for (int ks = 0; ks < TH_KC / 4; ks++) {
            double b1[NT], b2[NT];
#pragma unroll
            for (int b = 0; b < NT; b++) {
                const int kk = (ng * NT + b) * 4 + kq;
                const double x = bs[brow(arrX, ks * 4 + t) + kk];
                if (CPLX) {
                    const double y = ysgn * bs[brow(arrY, ks * 4 + t) + kk];      // m = 0: the b_0 rows are zero-filled, y = 0
                    b1[b] = fma(x, xscl, y);
                    b2[b] = fma(x, xscl, -y);
                } else {
                    b1[b] = x;
                }
            }
#pragma unroll
            for (int a = 0; a < MT; a++) {
                const double a1 = as[a * 8 * TH_PA + ks * 4];
#pragma unroll
                for (int b = 0; b < NT; b++) dmma(acc[0][a][b][0], acc[0][a][b][1], a1, b1[b]);
                if (CPLX) {
                    const double a2 = as[(Nt8c + a * 8) * TH_PA + ks * 4];
#pragma unroll
                    for (int b = 0; b < NT; b++) dmma(acc[NMAT - 1][a][b][0], acc[NMAT - 1][a][b][1], a2, b2[b]);
                }
            }
        }
    }
    // epilogue: lane owns latitude i = r0 + (mg*MT + a)*8 + g and radius k = k0 + (ng*NT + b)*4 + t; 32-bit offsets from one base
    double *Ro = cout + (size_t)cmp.dof * dofsz + (size_t)mca * vec + k0;       // a~_m row block of the (real part of the) component
    const int eAB = (int)offAB, eRI = (int)dofsz;                               // a dof array is far below 2^31 elements
#pragma unroll
    for (int a = 0; a < MT; a++) {
        const int i = r0 + (mg * MT + a) * 8 + g;
        if (i >= Nt) continue;
#pragma unroll
        for (int b = 0; b < NT; b++) {
            const int kl = (ng * NT + b) * 4 + t;
            if (kl >= nrad) continue;
            const int off = i * Nr + kl;
            const double pp = acc[0][a][b][0], qq = acc[0][a][b][1];
            if (!CPLX) {
                Ro[off] = pp;
                if (m > 0) Ro[off + eAB] = qq;
            } else if (m > 0) {
                const double ss = acc[NMAT - 1][a][b][0], tt = acc[NMAT - 1][a][b][1];
                Ro[off] = pp + ss;
                Ro[off + eAB] = tt - qq;
                Ro[off + eRI] = qq + tt;
                Ro[off + eRI + eAB] = pp - ss;
            } else {
                Ro[off] = pp;
                Ro[off + eRI] = qq;
            }
        }
    }
}

static inline size_t theta2_smem_bytes(int Nt8, bool cplx, int NT = 1, int kdim = 1 << 20) {      // NT = 1 has the larger tile; Nt8 = rows per CTA, kdim = padded K
    return (size_t)std::min(TH_STAGES, (kdim + TH_KC - 1) / TH_KC) * ((size_t)(cplx ? 2 : 1) * Nt8 * TH_PA + (cplx ? 4 : 2) * TH_ARR_OF(NT)) * sizeof(double);
}

// ---------------------------------------------------------------------------------------------
// EQUATORIAL FOLD of the theta step for real components (n = 0).  The Gauss latitudes (eq. 3) are symmetric about the
// equator and sY_lm(pi - theta) = (-1)^(l+m) (-s)Y_lm(theta), so with i' = Ntheta - 1 - i the filter matrices satisfy
// F^{-n}_m[i'][k'] = F^n_m[i][k] (tests/test_host_matrices.py); F^0_m is centrosymmetric.  With h = Ntheta / 2 and, for k < h,
//     xE[k] = x[k] + x[k'],   xO[k] = x[k] - x[k'],     G+-[i][k] = (F^0_m[i][k] +- F^0_m[i][k']) / 2      (h x h, built on the host)
// the same sums regroup to   y[i] = (G+ xE)[i] + (G- xO)[i],   y[i'] = (G+ xE)[i] - (G- xO)[i]:
// two (Ntheta/2)^2 products instead of one Ntheta^2 -- half the DMMAs, the regrouping of the two reflection folds already in
// the path (d/dtheta: antipodal planes, Fourier transforms: phi -> 2 pi - phi).  Requires Ntheta even.
// Data flow = the complex path of k_theta2: two matrices (G+, G-), four staged row sets (a_m top, a_m bottom reversed, b_m top,
// b_m bottom reversed), fragments b1 = top + bottom, b2 = top - bottom, lane-local epilogue.  G: [2][L+1][h8][h8] zero padded.
// ---------------------------------------------------------------------------------------------
template <int MT, int NT>
__global__ void __launch_bounds__(NT == 3 ? 384 : 896, 1)
k_theta_fold(ThetaBatch2 comps, const double *__restrict__ G, int L, int Nt, int h8, int Nr, int MC4, int mgroups,
             const double *__restrict__ coef, double *__restrict__ cout) {
    extern __shared__ __align__(16) double sm[];
    constexpr int TH_PKB = TH_PKB_OF(NT), TH_ARR = TH_ARR_OF(NT);
    const ThetaComp2 cmp = comps.c[blockIdx.y];
    const int m = blockIdx.x, k0 = blockIdx.z * TH_RC, h = Nt >> 1;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int mg = warp % mgroups, ng = warp / mgroups, nwarps = blockDim.x >> 5;
    const size_t vec = (size_t)Nt * Nr, dofsz = (size_t)MC4 * vec, gsz = (size_t)h8 * h8;
    const int stageA = 2 * h8 * TH_PA, stageB = 4 * TH_ARR;
    // row sets: arr = 2 * (0: a_m, 1: b_m) + (0: top rows ascending, 1: bottom rows descending); the sets a lane pair (v = 0, 1)
    // reads together (arr 0 and 2, arr 1 and 3) are neighbours in the NT = 1 layout
    auto brow = [&](int arr, int r) {
        const int slot = (arr == 0) ? 0 : (arr == 2) ? 1 : (arr == 1) ? 2 : 3;
        return NT == 1 ? slot * TH_ARR + r * TH_PKB : (arr * TH_KC + r) * TH_PKB;
    };
    double *As = sm, *Bs = sm + min(TH_STAGES, (h8 + TH_KC - 1) / TH_KC) * stageA;
    const int nrad = min(TH_RC, Nr - k0);
    const double *G0 = G + (size_t)m * gsz;
    const long dG = (long)(L + 1) * (long)gsz;                                  // G- relative to G+
    const int nchunks = (h8 + TH_KC - 1) / TH_KC;
    const int hF = tid & 7, rF0 = tid >> 3, rFstep = blockDim.x >> 3;
    const size_t offAB = (size_t)L * vec;                                       // b_m relative to a_m
    const double *srcA = coef + (size_t)cmp.dof * dofsz + (size_t)m * vec + k0 + lane;
    const bool live0 = lane < nrad, live1 = lane + 32 < nrad, lane_hi = lane < TH_RC - 32;
    auto load_chunk = [&](int kc, int st) {
        double *as = As + st * stageA + rF0 * TH_PA + 2 * hF;
        if (kc * TH_KC + 2 * hF < h8) {
            const double *fs = G0 + rF0 * h8 + kc * TH_KC + 2 * hF;
            const int fstep = rFstep * h8;
#pragma unroll 1
            for (int r = rF0; r < h8; r += rFstep, as += rFstep * TH_PA, fs += fstep) {
                cp_async16(as, fs);
                cp_async16(as + h8 * TH_PA, fs + dG);
            }
        } else {
#pragma unroll 1
            for (int r = rF0; r < h8; r += rFstep, as += rFstep * TH_PA) {
                as[0] = 0.0; as[1] = 0.0;
                as[h8 * TH_PA] = 0.0; as[h8 * TH_PA + 1] = 0.0;
            }
        }
        const int kbase = kc * TH_KC;
        double *bs = Bs + st * stageB + lane;
        const int gstep = nwarps * Nr, sstep = nwarps * TH_PKB;
#pragma unroll
        for (int arr = 0; arr < 4; arr++) {
            const bool bot = arr & 1;
            const double *gp = srcA + (arr >> 1) * offAB + (size_t)(bot ? Nt - 1 - (kbase + warp) : kbase + warp) * Nr;
            double *sp = bs + brow(arr, warp);
            const bool arrdead = (m == 0) && (arr >> 1);                                // b_0 does not exist
#pragma unroll 1
            for (int r = warp; r < TH_KC; r += nwarps, sp += sstep) {
                const bool dead = arrdead || kbase + r >= h;
                const double *gq = dead ? srcA : gp;                                    // dead rows: any valid address (not read)
                cp_async8_ign(sp, gq, dead || !live0);
                if (lane_hi) cp_async8_ign(sp + 32, gq + 32, dead || !live1);
                if (bot) gp -= gstep; else gp += gstep;
            }
        }
    };

    double acc[2][MT][NT][2];
#pragma unroll
    for (int x = 0; x < 2; x++)
#pragma unroll
        for (int a = 0; a < MT; a++)
#pragma unroll
            for (int b = 0; b < NT; b++) acc[x][a][b][0] = acc[x][a][b][1] = 0.0;
#pragma unroll
    for (int s = 0; s < TH_STAGES - 1; s++) {
        if (s < nchunks) load_chunk(s, s);
        cp_async_commit();
    }
    const int v = g & 1, kq = g >> 1;
    const int oX = brow(2 * v, t), oY = brow(2 * v + 1, t);
    for (int kc = 0; kc < nchunks; kc++) {
        cp_async_wait<TH_STAGES - 2>();
        __syncthreads();
        if (kc + TH_STAGES - 1 < nchunks) load_chunk(kc + TH_STAGES - 1, (kc + TH_STAGES - 1) % TH_STAGES);
        cp_async_commit();
        const double *as = As + (kc % TH_STAGES) * stageA + (mg * MT * 8 + g) * TH_PA + t;
        const double *bs = Bs + (kc % TH_STAGES) * stageB;
#pragma unroll
        for (int ks = 0; ks < TH_KC / 4; ks++) {
            double b1[NT], b2[NT];
#pragma unroll
            for (int b = 0; b < NT; b++) {
                const int kk = (ng * NT + b) * 4 + kq + ks * 4 * TH_PKB;
                const double x = bs[oX + kk], y = bs[oY + kk];
                b1[b] = x + y;
                b2[b] = x - y;
            }
#pragma unroll
            for (int a = 0; a < MT; a++) {
                const double a1 = as[a * 8 * TH_PA + ks * 4];
#pragma unroll
                for (int b = 0; b < NT; b++) dmma(acc[0][a][b][0], acc[0][a][b][1], a1, b1[b]);
                const double a2 = as[(h8 + a * 8) * TH_PA + ks * 4];
#pragma unroll
                for (int b = 0; b < NT; b++) dmma(acc[1][a][b][0], acc[1][a][b][1], a2, b2[b]);
            }
        }
    }
    // epilogue: lane owns the latitudes i = (mg*MT + a)*8 + g < h and i' = Ntheta - 1 - i, radius k = k0 + (ng*NT + b)*4 + t
    double *Ro = cout + (size_t)cmp.dof * dofsz + (size_t)m * vec + k0;
    const int eAB = (int)offAB;
#pragma unroll
    for (int a = 0; a < MT; a++) {
        const int i = (mg * MT + a) * 8 + g;
        if (i >= h) continue;
#pragma unroll
        for (int b = 0; b < NT; b++) {
            const int kl = (ng * NT + b) * 4 + t;
            if (kl >= nrad) continue;
            const int off = i * Nr + kl, offm = (Nt - 1 - i) * Nr + kl;
            const double p0 = acc[0][a][b][0], p1 = acc[0][a][b][1], s0 = acc[1][a][b][0], s1 = acc[1][a][b][1];
            Ro[off] = p0 + s0;
            Ro[offm] = p0 - s0;
            if (m > 0) { Ro[off + eAB] = p1 + s1; Ro[offm + eAB] = p1 - s1; }
        }
    }
}
static inline size_t theta_fold_smem_bytes(int h8, int NT) {
    return (size_t)std::min(TH_STAGES, (h8 + TH_KC - 1) / TH_KC) * ((size_t)2 * h8 * TH_PA + 4 * TH_ARR_OF(NT)) * sizeof(double);
}
