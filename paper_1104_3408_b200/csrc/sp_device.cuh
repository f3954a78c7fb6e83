// Shell object and device-side helpers shared by the kernels of libspshell.
#pragma once
#include "../../include/spshell.h"
#include "sp_internal.h"

#include <cuda_runtime.h>

struct sp_shell {
    int Nr, Nt, Np, L;
    double rin, rout;
    int Nr8, Nr4, Nt8, Nt4, MC, MC4, MC8, J8, PU;
    bool grad_split_ok = false;   // the split gradient (r-theta kernel first, d/dphi GEMM with fused chain rule) is usable
    int grad_nwarps = 6, grad3_nwarps = 6, num_sms = 148;
    int grad3_ctas[2] = {0, 0};      // same for the folded kernel k_grad_rtheta3
    int grad3_alt_nwarps = 0, grad3_alt_ctas = 0;   // narrower CTAs (4 warps) of the single-buffered k_grad_rtheta3 for small calls: more CTAs per SM, one round
    int grad_ctas[2] = {1, 0};       // resident CTAs per SM with NBUF = 1 / 2 (0: does not fit)
    size_t grad_smem[2] = {0, 0};
    int gradKT;                   // radial tiles per warp task of k_grad_rtheta2 (3 or 5)
    size_t npts;
    bool built, host_built;
    SpHostMatrices *host = nullptr;
    // device-resident tables (owned)
    double *d_cd = nullptr;        // CD^ [Nr8][PU], zero padded                       (eq. 9)
    double *d_g2 = nullptr;        // FD_{2Nt} circulant generator [2Nt]               (eq. 8)
    double *d_g3 = nullptr;        // FD_{Np}  circulant generator [Np]
    double *d_an = nullptr;        // Fourier analysis  [MC8][Np], zero padded rows    (eq. 24)
    double *d_sy = nullptr;        // Fourier synthesis [J8][MC4], zero padded         (eq. 23)
    double *d_F = nullptr;         // F^n_m [7][L+1][Nt8][Nt4], zero padded            (eq. 62)
    double *d_G = nullptr;         // equatorial fold of F^0_m: G+, G- [2][L+1][h8][h8], zero padded (Ntheta even; k_theta_fold)
    int h8 = 0;                    // Ntheta / 2 rounded up to 8
    // shared-memory-staged phi GEMM operands: rows padded to the warp tiling, K padded to 8, zero filled
    double *d_fd3p = nullptr;
    int fd3_MT = 0, fd3_mg = 0, fd3_Mpad = 0;
    int Np8 = 0;                  // K of d/dphi (Np) rounded up to 8
    // folded Fourier matrices (phi -> 2 pi - phi reflection, see k_pointwise): cosine / sine blocks of analysis and synthesis
    struct PhiMat { double *d = nullptr; int M = 0, K = 0, K8 = 0, MT = 0, mg = 0, Mpad = 0; };
    // folded d/dphi operator (k_phi_grad_fold): Gm, Gp [gf_Mpad][gf_lda]
    double *d_gm = nullptr, *d_gp = nullptr;
    int gf_Mpad = 0, gf_lda = 0, gf_mg = 0;
    bool gf_ok = false;
    int theta_NT = 0;             // k_theta2 variant chosen at build time: NT + 20 * (rsplit - 1), NT = 3 or 1 column tiles per warp, rsplit = 1 or 2 row blocks (3, 1, 23, 21; 0: generic kernel)
    PhiMat m_ac, m_as, m_sc, m_ss;   // analysis cos [L+1][J/2+1], sin [L][J/2-1]; synthesis cos [J/2+1][L+1], sin [J/2-1][L]
    // operands of the fused filter kernels (kernels_fused.cuh), zero padded: analysis Ac [f_Mp][f_ldc] (a_0..a_L over jj = 0..h),
    // As [f_Mp][f_lds] (b_1..b_L over q, jj = h-1-q); synthesis Sc, Ss [f_Jp][f_ldk] (rows jj = 0..h; Ss rows 0 and h are zero)
    double *d_fAc = nullptr, *d_fAs = nullptr, *d_fSc = nullptr, *d_fSs = nullptr;
    int f_Mp = 0, f_ldc = 0, f_lds = 0, f_Jp = 0, f_ldk = 0;
    double *d_inv_r = nullptr, *d_sin_t = nullptr, *d_cos_t = nullptr, *d_inv_sin_t = nullptr, *d_sin_p = nullptr,
           *d_cos_p = nullptr;     // Jacobian / triad factors                          (eq. 6, 51)
    // optional per-stage timing (sp_profile_enable): events recorded on the caller's stream
    mutable bool prof = false;
    mutable cudaEvent_t ev[9] = {};
    mutable bool ev_set[9] = {};
    mutable bool grad_swapped = false;
    // internal side stream: independent launches of one stage (real / complex theta products, ...) run concurrently,
    // forked from and joined to the caller's stream by events
    cudaStream_t aux = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;   // last gradient ran (r,theta) kernel first, then the d/dphi GEMM
};

// stage marks: 0 grad start, 1 after d/dphi, 2 after r-theta+chain rule, 3 filter start, 4 after projection,
// 5 after phi analysis, 6 after theta matrices, 7 after phi synthesis, 8 after recombination
static inline void sp_mark(const sp_shell *s, cudaStream_t st, int idx) {
    if (s->prof) { cudaEventRecord(s->ev[idx], st); s->ev_set[idx] = true; }
}
extern unsigned long long g_sp_launches;   // kernels launched by hot calls since load (host counter)

sp_status sp_configure_kernels(sp_shell *s);

// ---------------------------------------------------------------------------------------------
// FP64 tensor-core tile: D(8x8) += A(8x4) * B(4x8), SASS DMMA.8x8x4 (the only native FP64 MMA shape
// on sm_100a).  Fragment ownership for lane l, g = l>>2, t = l&3:
//     A[g][t]            (row-major 8x4)
//     B[t][g]            (4x8, "col" operand)
//     C[g][2t], C[g][2t+1]
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}
