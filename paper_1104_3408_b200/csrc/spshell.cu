// libspshell -- C ABI entry points and shell object (see include/spshell.h).
// Kernels live in kernels_*.cuh; the host matrix construction in host_build.cpp.
#include "../../include/spshell.h"
#include "sp_internal.h"
#include "sp_device.cuh"
#include "kernels_gemm2.cuh"
#include "kernels_gradphi.cuh"

#include <cuda_runtime.h>
#include <cstdint>

#include <cmath>
#include <cstdio>
#include <algorithm>
#include <cstring>
#include <cstdlib>
#include <new>

#define SP_CUDA(x)                                   \
    do {                                             \
        cudaError_t e_ = (x);                        \
        if (e_ != cudaSuccess) return SP_ERR_CUDA;   \
    } while (0)

unsigned long long g_sp_launches = 0;

static int round_up(int a, int b) { return (a + b - 1) / b * b; }

extern "C" const char *sp_status_string(sp_status s) {
    switch (s) {
        case SP_OK: return "SP_OK";
        case SP_ERR_INVALID_ARG: return "SP_ERR_INVALID_ARG";
        case SP_ERR_NOT_BUILT: return "SP_ERR_NOT_BUILT";
        case SP_ERR_ALLOC: return "SP_ERR_ALLOC";
        case SP_ERR_CUDA: return "SP_ERR_CUDA";
        case SP_ERR_UNSUPPORTED: return "SP_ERR_UNSUPPORTED";
        case SP_ERR_SCRATCH_LIMIT: return "SP_ERR_SCRATCH_LIMIT: the call needs more scratch than the 32 MiB static array of sp_tensor_filter_noalloc holds; use sp_tensor_filter with a workspace";
    }
    return "SP_ERR_?";
}

extern "C" sp_status sp_shell_create(int Nr, int Nt, int Np, double rin, double rout, int L, sp_shell **out) {
    if (!out) return SP_ERR_INVALID_ARG;
    *out = nullptr;
    if (Nr < 2 || Nt < 2 || Np != 2 * Nt) return SP_ERR_INVALID_ARG;          // eq. 5
    if (!(rin > 0) || !(rout > rin)) return SP_ERR_INVALID_ARG;
    if (L < 0 || L > Nt - 1) return SP_ERR_INVALID_ARG;
    sp_shell *s = new (std::nothrow) sp_shell();
    if (!s) return SP_ERR_ALLOC;
    s->Nr = Nr; s->Nt = Nt; s->Np = Np; s->L = L; s->rin = rin; s->rout = rout;
    s->Nr8 = round_up(Nr, 8); s->Nr4 = round_up(Nr, 4);
    s->Nt8 = round_up(Nt, 8); s->Nt4 = round_up(Nt, 4);
    s->MC = 2 * L + 1; s->MC4 = round_up(s->MC, 4); s->MC8 = round_up(s->MC, 8);
    s->J8 = round_up(Np, 8);
    {   // radial tiling of the (r,theta) kernel and the shared-memory pitch (= 4 mod 8: conflict-free fragments)
        const int ktiles = s->Nr8 / 8;
        s->gradKT = (ktiles % 3 != 0 && ktiles % 5 == 0) ? 5 : 3;
        if (const char *e = getenv("SP_GRAD_KT")) { if (atoi(e) == 3 || atoi(e) == 5) s->gradKT = atoi(e); }   // tuning override
        s->PU = (ktiles + s->gradKT - 1) / s->gradKT * s->gradKT * 8 + 4;
    }
    s->npts = (size_t)Nr * Nt * Np;
    s->built = false; s->host_built = false;
    *out = s;
    return SP_OK;
}

static void free_dev(sp_shell *s) {
    double **p[] = {&s->d_cd, &s->d_g2, &s->d_g3, &s->d_an, &s->d_sy, &s->d_F, &s->d_G, &s->d_fd3p, &s->d_gm, &s->d_gp, &s->m_ac.d, &s->m_as.d, &s->m_sc.d, &s->m_ss.d, &s->d_fAc, &s->d_fAs, &s->d_fSc, &s->d_fSs, &s->d_inv_r, &s->d_sin_t, &s->d_cos_t,
                    &s->d_inv_sin_t, &s->d_sin_p, &s->d_cos_p};
    for (auto q : p) {
        if (*q) cudaFree(*q);
        *q = nullptr;
    }
}

extern "C" sp_status sp_shell_destroy(sp_shell *s) {
    if (!s) return SP_ERR_INVALID_ARG;
    free_dev(s);
    for (int q = 0; q < 9; q++)
        if (s->ev[q]) cudaEventDestroy(s->ev[q]);
    if (s->ev_fork) cudaEventDestroy(s->ev_fork);
    if (s->ev_join) cudaEventDestroy(s->ev_join);
    if (s->aux) cudaStreamDestroy(s->aux);
    delete s->host;
    delete s;
    return SP_OK;
}

static sp_status upload(double **dst, const double *src, size_t n) {
    SP_CUDA(cudaMalloc((void **)dst, n * sizeof(double)));
    SP_CUDA(cudaMemcpy(*dst, src, n * sizeof(double), cudaMemcpyHostToDevice));
    return SP_OK;
}

extern "C" sp_status sp_build_matrices(sp_shell *s) {
    if (!s) return SP_ERR_INVALID_ARG;
    s->built = false;
    delete s->host;
    s->host = new (std::nothrow) SpHostMatrices();
    if (!s->host) return SP_ERR_ALLOC;
    SpHostMatrices &H = *s->host;
    sp_host_build(s->Nr, s->Nt, s->Np, s->rin, s->rout, s->L, H);
    s->host_built = true;                      // sp_get_matrix works from here on (host logic is testable)
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return SP_ERR_CUDA;   // no CPU fallback for the hot path
    free_dev(s);
    const int Nr = s->Nr, Nt = s->Nt, Np = s->Np, L = s->L;
    sp_status st;
    // CD^ padded [Nr8][PU], zeros outside
    {
        std::vector<double> t((size_t)s->Nr8 * s->PU, 0.0);
        for (int i = 0; i < Nr; i++)
            for (int j = 0; j < Nr; j++) t[(size_t)i * s->PU + j] = H.cd[(size_t)i * Nr + j];
        if ((st = upload(&s->d_cd, t.data(), t.size())) != SP_OK) return st;
    }
    if ((st = upload(&s->d_g2, H.g2.data(), H.g2.size())) != SP_OK) return st;
    if ((st = upload(&s->d_g3, H.g3.data(), H.g3.size())) != SP_OK) return st;
    {   // analysis [MC8][Np], synthesis [J8][MC4]
        std::vector<double> a((size_t)s->MC8 * Np, 0.0), y((size_t)s->J8 * s->MC4, 0.0);
        for (int m = 0; m < s->MC; m++)
            for (int j = 0; j < Np; j++) a[(size_t)m * Np + j] = H.an[(size_t)m * Np + j];
        for (int j = 0; j < Np; j++)
            for (int m = 0; m < s->MC; m++) y[(size_t)j * s->MC4 + m] = H.sy[(size_t)j * s->MC + m];
        if ((st = upload(&s->d_an, a.data(), a.size())) != SP_OK) return st;
        if ((st = upload(&s->d_sy, y.data(), y.size())) != SP_OK) return st;
    }
    {   // F [7][L+1][Nt8][Nt8]
        std::vector<double> f((size_t)7 * (L + 1) * s->Nt8 * s->Nt8, 0.0);
        for (int q = 0; q < 7 * (L + 1); q++)
            for (int i = 0; i < Nt; i++)
                for (int j = 0; j < Nt; j++)
                    f[((size_t)q * s->Nt8 + i) * s->Nt8 + j] = H.F[((size_t)q * Nt + i) * Nt + j];
        if ((st = upload(&s->d_F, f.data(), f.size())) != SP_OK) return st;
    }
    s->h8 = 0;
    if (Nt % 2 == 0) {   // equatorial fold of F^0_m (k_theta_fold): G+- [i][k] = (F[i][k] +- F[i][Nt-1-k]) / 2, i, k < Nt / 2
        const int h = Nt / 2, h8 = (h + 7) / 8 * 8;
        std::vector<double> gf((size_t)2 * (L + 1) * h8 * h8, 0.0);
        for (int m = 0; m <= L; m++) {
            const double *F0 = H.F.data() + ((size_t)(3 * (L + 1) + m) * Nt) * Nt;
            for (int i = 0; i < h; i++)
                for (int k = 0; k < h; k++) {
                    const double a = F0[(size_t)i * Nt + k], b = F0[(size_t)i * Nt + (Nt - 1 - k)];
                    gf[(((size_t)m) * h8 + i) * h8 + k] = 0.5 * (a + b);
                    gf[(((size_t)(L + 1) + m) * h8 + i) * h8 + k] = 0.5 * (a - b);
                }
        }
        if ((st = upload(&s->d_G, gf.data(), gf.size())) != SP_OK) return st;
        s->h8 = h8;
    }
    {   // padded operands of k_phi_gemm: FD_{Np}, and the folded Fourier blocks (entries taken from H.an / H.sy)
        PhiTiling t1 = phi_tiling(Np);
        s->fd3_MT = t1.MT; s->fd3_mg = t1.mgroups; s->fd3_Mpad = t1.Mpad;
        s->Np8 = round_up(Np, PG_KC);
        std::vector<double> a((size_t)t1.Mpad * s->Np8, 0.0);
        for (int i = 0; i < Np; i++)
            for (int j = 0; j < Np; j++) a[(size_t)i * s->Np8 + j] = H.g3[((i - j) % Np + Np) % Np];
        if ((st = upload(&s->d_fd3p, a.data(), a.size())) != SP_OK) return st;
        {   // folded d/dphi operator: Gm[j'][jj] = g(j'-jj) - g(j'+jj), Gp[j'][jj] = g(j'-jj) + g(j'+jj) (ends: g(j'), g(j'-h))
            const int hh = Np / 2, M = hh + 1, mt = (M + 7) / 8;
            s->gf_mg = (mt + 3) / 4; s->gf_Mpad = s->gf_mg * 32; s->gf_lda = round_up(M, 8);
            auto gg = [&](int d) { return H.g3[((d % Np) + Np) % Np]; };
            std::vector<double> gm((size_t)s->gf_Mpad * s->gf_lda, 0.0), gp(gm.size(), 0.0);
            for (int jp = 0; jp < M; jp++)
                for (int jj = 0; jj < M; jj++) {
                    const bool end = (jj == 0 || jj == hh);
                    gm[(size_t)jp * s->gf_lda + jj] = end ? 0.0 : gg(jp - jj) - gg(jp + jj);
                    gp[(size_t)jp * s->gf_lda + jj] = end ? gg(jp - jj) : gg(jp - jj) + gg(jp + jj);
                }
            if ((st = upload(&s->d_gm, gm.data(), gm.size())) != SP_OK) return st;
            if ((st = upload(&s->d_gp, gp.data(), gp.size())) != SP_OK) return st;
        }
        const int MC = s->MC, h = Nt;                 // h = J/2
        auto mk = [&](sp_shell::PhiMat &pm, int M, int K, auto entry) -> sp_status {
            PhiTiling tl = phi_tiling(M > 0 ? M : 1);
            pm.M = M; pm.K = K; pm.K8 = round_up(K > 0 ? K : 1, PG_KC); pm.MT = tl.MT; pm.mg = tl.mgroups; pm.Mpad = tl.Mpad;
            std::vector<double> v((size_t)pm.Mpad * pm.K8, 0.0);
            for (int r = 0; r < M; r++)
                for (int c = 0; c < K; c++) v[(size_t)r * pm.K8 + c] = entry(r, c);
            return upload(&pm.d, v.data(), v.size());
        };
        // rows of H.an: 0 = a_0, 2m-1 = a_m, 2m = b_m; columns of H.sy likewise
        if ((st = mk(s->m_ac, L + 1, h + 1, [&](int m, int j) { return H.an[(size_t)(m == 0 ? 0 : 2 * m - 1) * Np + j]; })) != SP_OK) return st;
        if ((st = mk(s->m_as, L, h - 1, [&](int r, int c) { return H.an[(size_t)(2 * (r + 1)) * Np + (c + 1)]; })) != SP_OK) return st;
        if ((st = mk(s->m_sc, h + 1, L + 1, [&](int j, int m) { return H.sy[(size_t)j * MC + (m == 0 ? 0 : 2 * m - 1)]; })) != SP_OK) return st;
        if ((st = mk(s->m_ss, h - 1, L, [&](int r, int c) { return H.sy[(size_t)(r + 1) * MC + 2 * (c + 1)]; })) != SP_OK) return st;
        {   // operands of the fused kernels (kernels_fused.cuh): same entries, their own padding
            s->f_Mp = round_up(L + 1, 8); s->f_ldc = round_up(h + 1, 16); s->f_lds = round_up(std::max(h - 1, 1), 16);
            s->f_Jp = round_up(h + 1, 8); s->f_ldk = round_up(L + 1, 16);
            std::vector<double> ac((size_t)s->f_Mp * s->f_ldc, 0.0), as((size_t)s->f_Mp * s->f_lds, 0.0);
            std::vector<double> sc((size_t)s->f_Jp * s->f_ldk, 0.0), ss(sc.size(), 0.0);
            for (int m = 0; m <= L; m++)
                for (int jj = 0; jj <= h; jj++) {
                    ac[(size_t)m * s->f_ldc + jj] = H.an[(size_t)(m == 0 ? 0 : 2 * m - 1) * Np + jj];
                    sc[(size_t)jj * s->f_ldk + m] = H.sy[(size_t)jj * MC + (m == 0 ? 0 : 2 * m - 1)];
                }
            for (int m = 1; m <= L; m++)
                for (int jj = 1; jj <= h - 1; jj++) {
                    as[(size_t)(m - 1) * s->f_lds + (h - 1 - jj)] = H.an[(size_t)(2 * m) * Np + jj];
                    ss[(size_t)jj * s->f_ldk + (m - 1)] = H.sy[(size_t)jj * MC + 2 * m];
                }
            if ((st = upload(&s->d_fAc, ac.data(), ac.size())) != SP_OK) return st;
            if ((st = upload(&s->d_fAs, as.data(), as.size())) != SP_OK) return st;
            if ((st = upload(&s->d_fSc, sc.data(), sc.size())) != SP_OK) return st;
            if ((st = upload(&s->d_fSs, ss.data(), ss.size())) != SP_OK) return st;
        }
    }
    if ((st = upload(&s->d_inv_r, H.inv_r.data(), Nr)) != SP_OK) return st;
    if ((st = upload(&s->d_sin_t, H.sin_t.data(), Nt)) != SP_OK) return st;
    if ((st = upload(&s->d_cos_t, H.cos_t.data(), Nt)) != SP_OK) return st;
    if ((st = upload(&s->d_inv_sin_t, H.inv_sin_t.data(), Nt)) != SP_OK) return st;
    if ((st = upload(&s->d_sin_p, H.sin_p.data(), Np)) != SP_OK) return st;
    if ((st = upload(&s->d_cos_p, H.cos_p.data(), Np)) != SP_OK) return st;
    if (!s->aux) {
        SP_CUDA(cudaStreamCreateWithFlags(&s->aux, cudaStreamNonBlocking));
        SP_CUDA(cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming));
        SP_CUDA(cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming));
    }
    if ((st = sp_configure_kernels(s)) != SP_OK) return st;
    s->built = true;
    return SP_OK;
}

extern "C" sp_status sp_get_matrix(const sp_shell *s, int which, int n, int m, double *out, int *rows, int *cols) {
    if (!s) return SP_ERR_INVALID_ARG;
    if (!s->host_built) return SP_ERR_NOT_BUILT;
    const SpHostMatrices &H = *s->host;
    const int Nr = s->Nr, Nt = s->Nt, Np = s->Np, L = s->L, MC = s->MC;
    int r = 0, c = 0;
    switch (which) {
        case 0: r = c = Nr; break;
        case 1: r = Nt; c = 2 * Nt; break;
        case 2: r = c = Np; break;
        case 3: r = MC; c = Np; break;
        case 4: r = Np; c = MC; break;
        case 5:
            if (n < -3 || n > 3 || m < 0 || m > L) return SP_ERR_INVALID_ARG;
            r = c = Nt; break;
        default: return SP_ERR_INVALID_ARG;
    }
    if (rows) *rows = r;
    if (cols) *cols = c;
    if (!out) return SP_OK;
    switch (which) {
        case 0: memcpy(out, H.cd.data(), sizeof(double) * r * c); break;
        case 1:
            for (int i = 0; i < r; i++)
                for (int j = 0; j < c; j++) out[(size_t)i * c + j] = H.g2[((i - j) % c + c) % c];
            break;
        case 2:
            for (int i = 0; i < r; i++)
                for (int j = 0; j < c; j++) out[(size_t)i * c + j] = H.g3[((i - j) % c + c) % c];
            break;
        case 3: memcpy(out, H.an.data(), sizeof(double) * r * c); break;
        case 4: memcpy(out, H.sy.data(), sizeof(double) * r * c); break;
        case 5: memcpy(out, &H.F[((size_t)(n + 3) * (L + 1) + m) * Nt * Nt], sizeof(double) * r * c); break;
    }
    return SP_OK;
}

// =================================================================================================
// Hot calls
// =================================================================================================
#include "kernels_gemm.cuh"
#include "kernels_grad.cuh"
#include "kernels_filter.cuh"
#include "kernels_theta2.cuh"
#include "kernels_fused.cuh"
#include "kernels_wave.cuh"
#include "kernels_ghg.cuh"

// fork the side stream off the caller's stream / join it back (events; capture-safe; no host synchronisation)
static bool sp_fork(const sp_shell *s, cudaStream_t st) {
    return s->aux && cudaEventRecord(s->ev_fork, st) == cudaSuccess && cudaStreamWaitEvent(s->aux, s->ev_fork, 0) == cudaSuccess;
}
static bool sp_join(const sp_shell *s, cudaStream_t st) {
    return cudaEventRecord(s->ev_join, s->aux) == cudaSuccess && cudaStreamWaitEvent(st, s->ev_join, 0) == cudaSuccess;
}

// smallest Nphi at which d/dphi runs reflection-folded (k_phi_grad_fold); SP_DPHI_FOLD_MIN overrides (experiments)
static int sp_dphi_fold_min() {
    static const int v = [] { const char *e = getenv("SP_DPHI_FOLD_MIN"); return e ? atoi(e) : 128; }();
    return v;
}

// theta step launcher.  Variant code v = NT + 20 * (rsplit - 1): NT = 3 or 1 column tiles per warp, rsplit = 1 or 2 row blocks
// per (component, m, radial block) (see kernels_theta2.cuh): 3, 1, 23, 21
static inline int th_NT(int v) { return v % 20; }
static inline int th_rsplit(int v) { return v / 20 + 1; }
static void theta2_tiling(const sp_shell *s, int v, int &MT, int &mgroups) {
    const int NT = th_NT(v), mtiles = s->Nt8 / 8 / th_rsplit(v), ngc = 9 / NT;
    MT = (mtiles % 3 == 0) ? 3 : (mtiles % 4 == 0) ? 4 : (mtiles < 3 ? mtiles : 3);
    if (((mtiles + MT - 1) / MT) * ngc > (NT == 3 ? 12 : 28) && mtiles % 4 == 0) MT = 4;
    mgroups = (mtiles + MT - 1) / MT;
}
static bool theta2_fits(const sp_shell *s, int v) {
    const int NT = th_NT(v), rs = th_rsplit(v);
    if ((s->Nt8 / 8) % rs != 0 || s->Nt8 / rs < 8) return false;
    int MT, mg;
    theta2_tiling(s, v, MT, mg);
    return mg * (9 / NT) <= (NT == 3 ? 12 : 28) && theta2_smem_bytes(s->Nt8 / rs, true, NT, s->Nt8) <= 227 * 1024;      // launch bounds of k_theta2
}
static sp_status launch_theta2(const sp_shell *s, int v, const std::vector<ThetaComp2> &rl, const std::vector<ThetaComp2> &cx,
                               const double *coef1, double *coef2, cudaStream_t st) {
    const int NT = th_NT(v), rsplit = th_rsplit(v);
    int MT, mgroups;
    theta2_tiling(s, v, MT, mgroups);
    const dim3 block(mgroups * (9 / NT) * 32);
    const int gz = (s->Nr + TH_RC - 1) / TH_RC;
    // the real and the complex components are independent: the (shorter) real launch runs on the side stream, so CTAs of
    // different lengths share the SMs (no lock-step fill/drain phases) and each launch fills the other's tail
    const bool fork = s->aux && !rl.empty() && !cx.empty();
    cudaStream_t main_st = st;
    if (fork) {
        if (cudaEventRecord(s->ev_fork, main_st) != cudaSuccess || cudaStreamWaitEvent(s->aux, s->ev_fork, 0) != cudaSuccess) return SP_ERR_CUDA;
    }
    // real components: equatorially folded kernel (half the DMMAs) when Ntheta is even; SP_THETA_FOLD=0 switches it off (experiments)
    static const bool fold_env = [] { const char *e = getenv("SP_THETA_FOLD"); return !e || atoi(e) != 0; }();
    int fMT = 0, fmg = 0;
    if (s->d_G && fold_env) {
        const int mt = s->h8 / 8;
        fMT = (mt % 3 == 0) ? 3 : (mt % 4 == 0) ? 4 : (mt < 3 ? mt : (mt % 2 == 0 ? 2 : 1));
        fmg = mt / fMT;
        if (fmg * (9 / NT) > (NT == 3 ? 12 : 28) || theta_fold_smem_bytes(s->h8, NT) > 227 * 1024) fMT = 0;
    }
    for (int pass = 1; pass >= 0; pass--) {
        const std::vector<ThetaComp2> &lst = pass ? cx : rl;
        st = (fork && pass == 0) ? s->aux : main_st;
        if (pass == 0 && fMT > 0) {
            const size_t smf = theta_fold_smem_bytes(s->h8, NT);
            const dim3 fblock(fmg * (9 / NT) * 32);
            for (size_t c0 = 0; c0 < lst.size(); c0 += SP_THETA2_BATCH) {
                ThetaBatch2 b;
                const int nb = (int)std::min<size_t>(SP_THETA2_BATCH, lst.size() - c0);
                for (int q = 0; q < nb; q++) b.c[q] = lst[c0 + q];
                const dim3 grid(s->L + 1, nb, gz);
#define SP_THF(MTV, NTV) k_theta_fold<MTV, NTV><<<grid, fblock, smf, st>>>(b, s->d_G, s->L, s->Nt, s->h8, s->Nr, s->MC4, fmg, coef1, coef2);
#define SP_THFM(NTV) switch (fMT) { case 1: SP_THF(1, NTV) break; case 2: SP_THF(2, NTV) break; case 3: SP_THF(3, NTV) break; default: SP_THF(4, NTV) break; }
                if (NT == 3) { SP_THFM(3) } else { SP_THFM(1) }
#undef SP_THFM
#undef SP_THF
                g_sp_launches += 1;
            }
            continue;
        }
        const size_t sm = theta2_smem_bytes(s->Nt8 / rsplit, pass == 1, NT, s->Nt8);
        for (size_t c0 = 0; c0 < lst.size(); c0 += SP_THETA2_BATCH) {
            ThetaBatch2 b;
            const int nb = (int)std::min<size_t>(SP_THETA2_BATCH, lst.size() - c0);
            for (int q = 0; q < nb; q++) b.c[q] = lst[c0 + q];
            const int sfast = (rsplit > 1 && (double)nb * (pass ? 2 : 1) * s->MC * s->Nt * s->Nr * sizeof(double) > SP_SPLIT_FAST_BYTES) ? 1 : 0;
            const dim3 grid = sfast ? dim3((s->L + 1) * rsplit, nb, gz) : dim3(s->L + 1, nb, gz * rsplit);
#define SP_TH2(MTV, NTV)                                                                                                        \
    if (pass) k_theta2<MTV, NTV, true><<<grid, block, sm, st>>>(b, s->d_F, s->L, s->Nt, s->Nt8, s->Nr, s->MC4, mgroups, rsplit, coef1, coef2, sfast); \
    else k_theta2<MTV, NTV, false><<<grid, block, sm, st>>>(b, s->d_F, s->L, s->Nt, s->Nt8, s->Nr, s->MC4, mgroups, rsplit, coef1, coef2, sfast);
#define SP_TH2M(NTV)                                                                                     \
    switch (MT) { case 1: SP_TH2(1, NTV) break; case 2: SP_TH2(2, NTV) break; case 3: SP_TH2(3, NTV) break; default: SP_TH2(4, NTV) break; }
            if (NT == 3) { SP_TH2M(3) } else { SP_TH2M(1) }
#undef SP_TH2M
#undef SP_TH2
            g_sp_launches += 1;
        }
    }
    if (fork) {
        if (cudaEventRecord(s->ev_join, s->aux) != cudaSuccess || cudaStreamWaitEvent(main_st, s->ev_join, 0) != cudaSuccess) return SP_ERR_CUDA;
    }
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

static size_t grad_smem_bytes(const sp_shell *s) {
    return ((size_t)2 * s->Nt8 * s->PU + (size_t)s->Nr8 * s->PU + 2 * s->Nt) * sizeof(double);
}

// Dynamic shared memory opt-in: the attribute belongs to the FUNCTION, process wide, not to a shell, so every instantiation is
// opted in to the device maximum (227 KB) and a shell built later (smaller or larger) can never lower the cap of an earlier one.
static const int SP_SMEM_MAX = 227 * 1024;

sp_status sp_configure_kernels(sp_shell *s) {
    size_t sm = grad_smem_bytes(s);
    if (sm > 227 * 1024) return SP_ERR_UNSUPPORTED;       // (r,theta) plane pair must fit one SM's shared memory
    SP_CUDA(cudaFuncSetAttribute(k_grad_rtheta<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));
    SP_CUDA(cudaFuncSetAttribute(k_grad_rtheta<5>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));
    {   // persistent (r,theta) kernel: two configurations, planes double-buffered (NBUF = 2) or not
        const int itiles = s->Nt8 / 8, ktiles = s->Nr8 / 8, KT = s->gradKT;
        const int ntasks = 2 * ((itiles + 1) / 2) * ((ktiles + KT - 1) / KT);
        s->grad_nwarps = (KT == 3) ? std::min(ntasks, 12) : std::min(ntasks, 6);
        cudaDeviceProp prop;
        int dev = 0;
        SP_CUDA(cudaGetDevice(&dev));
        SP_CUDA(cudaGetDeviceProperties(&prop, dev));
        s->num_sms = prop.multiProcessorCount;
        for (int nb = 1; nb <= 2; nb++) {
            s->grad_smem[nb - 1] = grad2_smem_bytes(s->Nt, s->Nt8, s->Nr8, s->PU, KT, nb, s->grad_nwarps);
            s->grad_ctas[nb - 1] = 0;
        }
        if (s->grad_smem[0] > 227 * 1024) return SP_ERR_UNSUPPORTED;
#define SP_GR_ATTR(KT_, SPL_, NB_)                                                                                      \
    SP_CUDA(cudaFuncSetAttribute(k_grad_rtheta2<KT_, SPL_, NB_>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));                                                          \
    SP_CUDA(cudaFuncSetAttribute(k_grad_rtheta2<KT_, SPL_, NB_>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        SP_GR_ATTR(3, true, 1) SP_GR_ATTR(5, true, 1) SP_GR_ATTR(3, false, 1) SP_GR_ATTR(5, false, 1)
        SP_GR_ATTR(3, true, 2) SP_GR_ATTR(5, true, 2) SP_GR_ATTR(3, false, 2) SP_GR_ATTR(5, false, 2)
#undef SP_GR_ATTR
        // resident CTAs per SM of the persistent grid, asked from the occupancy calculator for the variant that will run
        for (int nb = 1; nb <= 2; nb++) {
            if (s->grad_smem[nb - 1] > 227 * 1024) continue;
            int occ = 0;
            const int thr = s->grad_nwarps * 32;
            if (KT == 3) {
                if (nb == 1) SP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_grad_rtheta2<3, true, 1>, thr, s->grad_smem[0]));
                else SP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_grad_rtheta2<3, true, 2>, thr, s->grad_smem[1]));
            } else {
                if (nb == 1) SP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_grad_rtheta2<5, true, 1>, thr, s->grad_smem[0]));
                else SP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_grad_rtheta2<5, true, 2>, thr, s->grad_smem[1]));
            }
            s->grad_ctas[nb - 1] = occ;
        }
        if (s->grad_ctas[0] <= 0) return SP_ERR_UNSUPPORTED;
        // folded variant (k_grad_rtheta3): warp task = (latitude tile, radial group)
        {
            const int nt3 = itiles * ((ktiles + KT - 1) / KT);
            s->grad3_nwarps = (KT == 3) ? std::min(nt3, 12) : std::min(nt3, 6);
            if (const char *e = getenv("SP_GRAD_NWARPS")) { const int w = atoi(e); if (w >= 1 && w <= (KT == 3 ? 12 : 6)) s->grad3_nwarps = std::min(nt3, w); }   // tuning override
            const int thr = s->grad3_nwarps * 32;
            for (int nb = 1; nb <= 2; nb++) {
                s->grad3_ctas[nb - 1] = 0;
                if (s->grad_smem[nb - 1] > 227 * 1024) continue;
                int occ = 0;
                const int smb = (int)s->grad_smem[nb - 1];
#define SP_G3P(KT_, NB_, PU_)                                                                                            \
    SP_CUDA(cudaFuncSetAttribute(k_grad_rtheta3<KT_, NB_, PU_>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));      \
    SP_CUDA(cudaFuncSetAttribute(k_grad_rtheta3<KT_, NB_, PU_>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));   \
    SP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_grad_rtheta3<KT_, NB_, PU_>, thr, smb));
#define SP_G3(KT_, NB_)                                                                      \
    if (KT_ == 5 && s->PU == 44) { SP_G3P(KT_, NB_, 44) }                                    \
    else if (KT_ == 3 && s->PU == 28) { SP_G3P(KT_, NB_, 28) }                               \
    else if (KT_ == 3 && s->PU == 76) { SP_G3P(KT_, NB_, 76) }                               \
    else { SP_G3P(KT_, NB_, 0) }
                if (KT == 3) { if (nb == 1) { SP_G3(3, 1) } else { SP_G3(3, 2) } }
                else { if (nb == 1) { SP_G3(5, 1) } else { SP_G3(5, 2) } }
#undef SP_G3
                s->grad3_ctas[nb - 1] = occ;
                // small calls (fewer items than resident 6-warp CTAs can take in one round): 4-warp CTAs, when they split the warp
                // tasks evenly, fit more CTAs per SM (config 5: 320 items, 3 x 148 slots instead of 2 x 148; (r,theta) 41 -> 36 us)
                if (nb == 1 && KT == 5 && nt3 > 4 && nt3 % 4 == 0 && s->grad3_nwarps == 6 && !getenv("SP_GRAD_NWARPS") && !getenv("SP_GRAD_CTAS")) {
                    int occ_main = occ;
                    {
                        const int thr = 4 * 32;
                        if (s->PU == 44) { SP_G3P(5, 1, 44) } else { SP_G3P(5, 1, 0) }
                    }
                    s->grad3_alt_nwarps = 4; s->grad3_alt_ctas = occ;
                    occ = occ_main;
                }
                if (const char *e = getenv("SP_GRAD_CTAS")) { const int c = atoi(e); if (c >= 1 && c < occ) s->grad3_ctas[nb - 1] = c; }   // tuning override: resident CTAs per SM
#undef SP_G3P
            }
        }
    }
    PhiTiling tmax = {6, 4, 4 * 6 * 8};
    const int pg = (int)phi_smem_bytes(tmax);
#define SP_PGA(MTV)                                                                                             \
    SP_CUDA(cudaFuncSetAttribute(k_phi_gemm<MTV, false, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX)); \
    SP_CUDA(cudaFuncSetAttribute(k_phi_gemm<MTV, false, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));
    SP_PGA(4) SP_PGA(5) SP_PGA(6)
#undef SP_PGA
    {
        const size_t gfs = gradfold_smem_bytes(s->gf_Mpad, s->Np);
        s->gf_ok = s->gf_mg >= 1 && s->gf_mg <= 4 && gfs <= 227 * 1024;
        if (s->gf_ok) {
            SP_CUDA(cudaFuncSetAttribute(k_phi_grad_fold<4, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));
            SP_CUDA(cudaFuncSetAttribute(k_phi_grad_fold<4, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));
        }
    }
    {
        PhiTiling tg = phi_tiling(s->Np);
        const size_t pgg = phi_smem_bytes(tg, s->Np);
        s->grad_split_ok = pgg <= 227 * 1024 && tg.mgroups <= 4;
        if (s->grad_split_ok) {
#define SP_PGA(MTV)                                                                                                  \
    SP_CUDA(cudaFuncSetAttribute(k_phi_gemm<MTV, true, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX)); \
    SP_CUDA(cudaFuncSetAttribute(k_phi_gemm<MTV, true, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));
            SP_PGA(4) SP_PGA(5) SP_PGA(6)
#undef SP_PGA
        }
    }
    s->theta_NT = 0;
    if (theta2_smem_bytes(s->Nt8, true) <= 227 * 1024) {
        const int t1 = (int)theta2_smem_bytes(s->Nt8, false), t2 = (int)theta2_smem_bytes(s->Nt8, true);
#define SP_TA(MTV, NTV)                                                                                           \
    SP_CUDA(cudaFuncSetAttribute(k_theta2<MTV, NTV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));    \
    SP_CUDA(cudaFuncSetAttribute(k_theta2<MTV, NTV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));
        SP_TA(1, 3) SP_TA(2, 3) SP_TA(3, 3) SP_TA(4, 3) SP_TA(1, 1) SP_TA(2, 1) SP_TA(3, 1) SP_TA(4, 1)
#undef SP_TA
        if (s->d_G) {
            const int tf3 = (int)theta_fold_smem_bytes(s->h8, 3), tf1 = (int)theta_fold_smem_bytes(s->h8, 1);
#define SP_TF(MTV)                                                                                                      \
    SP_CUDA(cudaFuncSetAttribute(k_theta_fold<MTV, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX)); \
    SP_CUDA(cudaFuncSetAttribute(k_theta_fold<MTV, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX));
            SP_TF(1) SP_TF(2) SP_TF(3) SP_TF(4)
#undef SP_TF
        }
        // Variant choice BY RULE (deterministic across processes, boxes and profilers): the table below is the outcome of timing
        // runs on B200 (config 3, Ntheta = 48: NT = 3 unsplit; config 5, 64: NT = 1 split; config 4, 96: NT = 3
        // split).  SP_THETA_NT forces a variant; SP_THETA_TUNE=1 re-runs the timing race on scratch data instead of the rule.
        const int cand[4] = {3, 1, 23, 21};
        bool ok[4];
        int nok = 0, only = 0;
        const char *env = getenv("SP_THETA_NT");
        const int forced = env ? atoi(env) : 0;
        for (int v = 0; v < 4; v++) {
            ok[v] = theta2_fits(s, cand[v]);
            if (ok[v]) { nok++; only = cand[v]; }
            if (ok[v] && forced == cand[v]) s->theta_NT = forced;
        }
        if (s->theta_NT == 0 && nok == 1) s->theta_NT = only;
        const char *tune = getenv("SP_THETA_TUNE");
        if (s->theta_NT == 0 && nok > 1 && !(tune && atoi(tune) == 1)) {
            const int want = (s->Nt8 >= 88) ? 23 : (s->Nt8 >= 56) ? 21 : 3;
            const int order[4] = {want, 3, 23, 21};
            for (int q = 0; q < 4 && s->theta_NT == 0; q++)
                for (int v = 0; v < 4; v++)
                    if (ok[v] && cand[v] == order[q]) { s->theta_NT = cand[v]; break; }
            if (s->theta_NT == 0) s->theta_NT = only;
        }
        if (s->theta_NT == 0 && nok > 1) {
            const size_t dofsz = (size_t)s->MC4 * s->Nt * s->Nr;
            double *scr = nullptr;
            const int nscr = 48;
            if (cudaMalloc((void **)&scr, 2 * nscr * dofsz * sizeof(double)) != cudaSuccess) { cudaGetLastError(); s->theta_NT = ok[0] ? 3 : only; return SP_OK; }
            SP_CUDA(cudaMemset(scr, 0, 2 * nscr * dofsz * sizeof(double)));
            std::vector<ThetaComp2> rl, cx;
            for (int q = 0; q < 12; q++) rl.push_back({q, 0});
            for (int q = 0; q < 18; q++) cx.push_back({12 + 2 * q, 1 + q % 3});
            cudaEvent_t e0, e1;
            SP_CUDA(cudaEventCreate(&e0)); SP_CUDA(cudaEventCreate(&e1));
            float best[4] = {1e30f, 1e30f, 1e30f, 1e30f};
            for (int rep = 0; rep < 4; rep++)
                for (int v = 0; v < 4; v++) {
                    if (!ok[v]) continue;
                    cudaEventRecord(e0);
                    launch_theta2(s, cand[v], rl, cx, scr, scr + nscr * dofsz, 0);
                    cudaEventRecord(e1);
                    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(scr); return SP_ERR_CUDA; }
                    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
                    if (rep > 0 && ms < best[v]) best[v] = ms;
                }
            cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(scr);
            int bv = -1;
            for (int v = 0; v < 4; v++) if (ok[v] && (bv < 0 || best[v] < best[bv])) bv = v;
            s->theta_NT = cand[bv];
        }
    }
    return SP_OK;
}

extern "C" sp_status sp_get_tuning(const sp_shell *s, int out[4]) {
    if (!s || !out) return SP_ERR_INVALID_ARG;
    if (!s->built) return SP_ERR_NOT_BUILT;
    out[0] = s->theta_NT;
    out[1] = s->gradKT;
    out[2] = (s->gf_ok && s->Np >= sp_dphi_fold_min()) ? 1 : 0;
    out[3] = (s->grad3_ctas[1] > 0) ? 2 : 1;
    return SP_OK;
}

extern "C" sp_status sp_workspace_bytes(const sp_shell *s, int nfields, size_t *grad, size_t *filter, size_t *wave) {
    if (!s || nfields < 0) return SP_ERR_INVALID_ARG;
    const size_t vec = (size_t)s->Nt * s->Nr;
    if (grad) *grad = (size_t)nfields * s->npts * sizeof(double);
    if (filter) *filter = (size_t)nfields * (s->npts + 2 * (size_t)s->MC4 * vec) * sizeof(double);
    if (wave) *wave = (size_t)(4 + 12) * s->npts * sizeof(double);
    return SP_OK;
}

extern "C" sp_status sp_cartesian_gradient(const sp_shell *s, const double *u, int nf, double *du, void *ws, size_t wsb,
                                           void *stream) {
    if (!s || nf < 0) return SP_ERR_INVALID_ARG;
    if (!s->built) return SP_ERR_NOT_BUILT;
    if (nf == 0) return SP_OK;                          // empty input: nothing to do (pointers may be null)
    if (!u || !du) return SP_ERR_INVALID_ARG;
    if (!ws || wsb < (size_t)nf * s->npts * sizeof(double)) return SP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int Nr = s->Nr, Nt = s->Nt, Np = s->Np;
    const long plane = (long)Nr * Nt;
    const int itiles = s->Nt8 / 8, ktiles = s->Nr8 / 8;
    GradParams p;
    p.Nr = Nr; p.Nt = Nt; p.Np = Np; p.PU = s->PU; p.Nr8 = s->Nr8; p.Nr4 = s->Nr4; p.Nt8 = s->Nt8;
    p.cd = s->d_cd; p.g2 = s->d_g2;
    p.inv_r = s->d_inv_r; p.sin_t = s->d_sin_t; p.cos_t = s->d_cos_t; p.inv_sin_t = s->d_inv_sin_t;
    p.sin_p = s->d_sin_p; p.cos_p = s->d_cos_p;
    p.u = u; p.dphi = nullptr; p.du = du; p.nf = nf; p.nitems = Nt * nf;
    const dim3 grid(Nt, nf);
    PhiTiling tl = {s->fd3_MT, s->fd3_mg, s->fd3_Mpad};
    sp_mark(s, st, 0);
    // ---- fast path: (r,theta)-plane kernel first (W -> du[x], d_z -> du[z]), then the d/dphi GEMM whose epilogue
    //      applies the chain rule (eq. 6).  Needs Ntheta % 4 == 0, even strides and 16-byte aligned buffers.
    const bool aligned = !(((uintptr_t)u | (uintptr_t)du) & 15) && !((plane | (long)s->npts) & 1);
    if (Nt % 4 == 0 && s->grad_split_ok && aligned) {
      // SP_GRAD_CHUNK = c > 0: run the two kernels over chunks of c fields, so that a chunk's input and its intermediate W (written
      // by the plane kernel into the d_x slot, re-read by the d/dphi epilogue) are still in the 126 MB L2 when the second kernel
      // runs.  Off by default: measured slower on B200 -- the persistent plane kernel loses its pipelining
      // on short item lists.
      static const int chunk_env = [] { const char *e = getenv("SP_GRAD_CHUNK"); return e ? atoi(e) : 0; }();
      const int nf_all = nf, chunk = (chunk_env > 0 && chunk_env < nf) ? chunk_env : nf;
      const double *u_all = u;
      double *du_all = du;
      for (int f0 = 0; f0 < nf_all; f0 += chunk) {
        const int nf = std::min(chunk, nf_all - f0);
        const double *u = u_all + (size_t)f0 * s->npts;
        double *du = du_all + (size_t)f0 * s->npts;
        p.u = u; p.du = du; p.nf = nf_all; p.nitems = Nt * nf;
        const int KT = s->gradKT;
        const int ntasks = 2 * ((itiles + 1) / 2) * ((ktiles + KT - 1) / KT);
        if (s->grad3_ctas[0] > 0) {      // folded theta derivative (k_grad_rtheta3)
            int nthr = s->grad3_nwarps * 32;
            const int nb = (s->grad3_ctas[1] > 0 && p.nitems >= 3 * s->num_sms * s->grad3_ctas[1]) ? 2 : 1;
            int ncta = std::min(p.nitems, s->num_sms * s->grad3_ctas[nb - 1]);
            const size_t smb = s->grad_smem[nb - 1];
            if (nb == 1 && s->grad3_alt_ctas > 0) {      // rounds of resident CTAs x passes of a CTA's warps over its tasks
                const int nt3 = itiles * ((ktiles + KT - 1) / KT);
                auto cost = [&](int ctas, int nw) { return ((p.nitems + s->num_sms * ctas - 1) / (s->num_sms * ctas)) * ((nt3 + nw - 1) / nw); };
                if (cost(s->grad3_alt_ctas, s->grad3_alt_nwarps) < cost(s->grad3_ctas[0], s->grad3_nwarps)) {
                    nthr = s->grad3_alt_nwarps * 32;
                    ncta = std::min(p.nitems, s->num_sms * s->grad3_alt_ctas);
                }
            }
#define SP_G3L(KT_, NB_)                                                                               \
    if (KT_ == 5 && s->PU == 44) k_grad_rtheta3<KT_, NB_, 44><<<ncta, nthr, smb, st>>>(p);             \
    else if (KT_ == 3 && s->PU == 28) k_grad_rtheta3<KT_, NB_, 28><<<ncta, nthr, smb, st>>>(p);        \
    else if (KT_ == 3 && s->PU == 76) k_grad_rtheta3<KT_, NB_, 76><<<ncta, nthr, smb, st>>>(p);        \
    else k_grad_rtheta3<KT_, NB_, 0><<<ncta, nthr, smb, st>>>(p);
            if (KT == 3) { if (nb == 2) { SP_G3L(3, 2) } else { SP_G3L(3, 1) } }
            else { if (nb == 2) { SP_G3L(5, 2) } else { SP_G3L(5, 1) } }
#undef SP_G3L
            (void)ntasks;
        } else {
#define SPLITV true
        // double-buffered planes pay off once every persistent CTA gets >= 3 items; small launches keep more CTAs per SM
        const int nthr = s->grad_nwarps * 32;
        const int nb = (s->grad_ctas[1] > 0 && p.nitems >= 3 * s->num_sms * s->grad_ctas[1]) ? 2 : 1;
        const int ncta = std::min(p.nitems, s->num_sms * s->grad_ctas[nb - 1]);
        const size_t smb = s->grad_smem[nb - 1];
#define SP_GR_LAUNCH2(KT_, NB_) k_grad_rtheta2<KT_, SPLITV, NB_><<<ncta, nthr, smb, st>>>(p)
        if (KT == 3) { if (nb == 2) SP_GR_LAUNCH2(3, 2); else SP_GR_LAUNCH2(3, 1); }
        else { if (nb == 2) SP_GR_LAUNCH2(5, 2); else SP_GR_LAUNCH2(5, 1); }
#undef SP_GR_LAUNCH2
        (void)ntasks;
#undef SPLITV
        }
        if (cudaGetLastError() != cudaSuccess) return SP_ERR_CUDA;
        sp_mark(s, st, 1);
        PhiGradEpi ge = {du + (size_t)nf_all * s->npts, (long)s->npts, s->d_inv_r, s->d_inv_sin_t, s->d_sin_p, s->d_cos_p, Nr};
        // the fold halves the DMMAs but doubles the rows each warp finishes; measured: it wins from Nphi = 128 upwards
        if (s->gf_ok && Np >= sp_dphi_fold_min()) {      // reflection-folded d/dphi with the chain rule in the epilogue
            // 32-column tiles for this kernel at every size (config 4: 0.97 -> 0.88 ms; small states use them anyway)
            static const int nc_env = [] { const char *e = getenv("SP_PHI_NC"); return e ? atoi(e) : 0; }();
            const int NC = (nc_env == 64) ? 64 : 32;
            const long ctas = (long)(((int)plane + NC - 1) / NC) * nf;
            // row blocks as in launch_phi_gemm: two CTAs of half the rows when the kernel has an even number of warp rows and many
            // column tiles (config 4: 1.17 -> 0.97 ms)
            static const int zenv = [] { const char *e = getenv("SP_PHI_MSPLIT"); return e ? atoi(e) : -1; }();
            int zs = (s->gf_mg % 2 == 0 && ctas >= 8L * s->num_sms) ? 2 : 1;
            if (ctas < 4L * s->num_sms) zs = s->gf_mg;      // small states: one warp row per CTA (config 5: d/dphi 39 -> 29 us)
            if (zenv >= 1) zs = (s->gf_mg % zenv == 0) ? zenv : 1;
            const int mgc = s->gf_mg / zs;
            const int sfast = (zs > 1 && (double)s->npts * nf * sizeof(double) > SP_SPLIT_FAST_BYTES) ? 1 : 0;
            const dim3 gridf = sfast ? dim3(zs, ((int)plane + NC - 1) / NC, nf) : dim3(((int)plane + NC - 1) / NC, nf, zs);
            const size_t smf = gradfold_smem_bytes(s->gf_Mpad / zs, s->Np, NC);
            if (NC == 32)
                k_phi_grad_fold<4, 32><<<gridf, mgc * 2 * 32, smf, st>>>(
                    s->d_gm, s->d_gp, s->gf_lda, Np, s->gf_Mpad, u, plane, (long)s->npts, du, ge.Y, (long)s->npts, (int)plane, ge, sfast);
            else
                k_phi_grad_fold<4, 64><<<gridf, mgc * 4 * 32, smf, st>>>(
                    s->d_gm, s->d_gp, s->gf_lda, Np, s->gf_Mpad, u, plane, (long)s->npts, du, ge.Y, (long)s->npts, (int)plane, ge, sfast);
            if (cudaGetLastError() != cudaSuccess) return SP_ERR_CUDA;
        } else {
            sp_status e = launch_phi_gemm(s->d_fd3p, s->Np8, Np, tl, Np, u, plane, (long)s->npts, du, plane, (long)s->npts, (int)plane, nf,
                                          st, s->num_sms, &ge);
            if (e != SP_OK) return e;
        }
        g_sp_launches += 2;
      }
        sp_mark(s, st, 2);
        s->grad_swapped = true;
        return SP_OK;
    }
    // ---- general path: d/dphi into the workspace, then the plane kernel finishes all three components
    s->grad_swapped = false;
    g_sp_launches += 2;
    double *dphi = (double *)ws;
    p.dphi = dphi;
    sp_status e = launch_phi_gemm(s->d_fd3p, s->Np8, Np, tl, Np, u, plane, (long)s->npts, dphi, plane, (long)s->npts, (int)plane, nf, st, s->num_sms);
    if (e == SP_ERR_UNSUPPORTED)   // odd strides: generic global-memory kernel
        e = launch_gemm_cols<true>(s->d_g3, Np, Np, Np, u, plane, (long)s->npts, dphi, plane, (long)s->npts, (int)plane, nf, st);
    if (e != SP_OK) return e;
    sp_mark(s, st, 1);
    if (Nt % 4 == 0) {
        const int KT = s->gradKT;
        const int ntasks = 2 * ((itiles + 1) / 2) * ((ktiles + KT - 1) / KT);
#define SPLITV false
        // double-buffered planes pay off once every persistent CTA gets >= 3 items; small launches keep more CTAs per SM
        const int nthr = s->grad_nwarps * 32;
        const int nb = (s->grad_ctas[1] > 0 && p.nitems >= 3 * s->num_sms * s->grad_ctas[1]) ? 2 : 1;
        const int ncta = std::min(p.nitems, s->num_sms * s->grad_ctas[nb - 1]);
        const size_t smb = s->grad_smem[nb - 1];
#define SP_GR_LAUNCH2(KT_, NB_) k_grad_rtheta2<KT_, SPLITV, NB_><<<ncta, nthr, smb, st>>>(p)
        if (KT == 3) { if (nb == 2) SP_GR_LAUNCH2(3, 2); else SP_GR_LAUNCH2(3, 1); }
        else { if (nb == 2) SP_GR_LAUNCH2(5, 2); else SP_GR_LAUNCH2(5, 1); }
#undef SP_GR_LAUNCH2
        (void)ntasks;
#undef SPLITV
    } else {   // Ntheta not a multiple of 4: generic kernel
        const int ntasks = 2 * itiles * ((ktiles + 4) / 5);
        k_grad_rtheta<5><<<grid, (ntasks < 16 ? ntasks : 16) * 32, grad_smem_bytes(s), st>>>(p);
    }
    sp_mark(s, st, 2);
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

// ---- tensor classification -------------------------------------------------------------------
static int classify(const sp_tensor_desc &d) {
    auto okdim = [](int x) { return x == 3 || x == 4; };
    switch (d.rank) {
        case 0: return TT_SCALAR;
        case 1:
            if (!okdim(d.index_dim[0])) return -1;
            return d.index_dim[0] == 3 ? TT_VEC3 : TT_VEC4;
        case 2:
            if (!okdim(d.index_dim[0]) || d.index_dim[0] != d.index_dim[1]) return -2;
            if (!((d.sym_first == 0 && d.sym_second == 1) || (d.sym_first == 1 && d.sym_second == 0))) return -2;
            return d.index_dim[0] == 3 ? TT_SYM3 : TT_SYM4;
        case 3:
            if (!okdim(d.index_dim[0]) || !okdim(d.index_dim[1]) || d.index_dim[1] != d.index_dim[2]) return -2;
            if (!((d.sym_first == 1 && d.sym_second == 2) || (d.sym_first == 2 && d.sym_second == 1))) return -2;
            if (d.index_dim[0] == 3) return d.index_dim[1] == 3 ? TT_R3_3_3 : TT_R3_3_4;
            return d.index_dim[1] == 3 ? TT_R3_4_3 : TT_R3_4_4;
    }
    return -1;
}
static int tt_ncomp(int tt) {
    static const int n[TT_COUNT] = {1, 3, 4, 6, 10, 18, 30, 24, 40};
    return n[tt];
}
// spin-weight components of a tensor type in dof order: appends (dof, n, cplx)
static void tt_components(int tt, int dof0, std::vector<ThetaComp> &out) {
    int d = dof0;
    auto real = [&]() { out.push_back({d, 0, 0}); d += 1; };
    auto cplx = [&](int n) { out.push_back({d, n, 1}); d += 2; };
    auto sym = [&](int D, int shift, bool only_complex, bool as_complex_real) {
        int nreal = (D == 4) ? 4 : 2;
        if (!only_complex)
            for (int q = 0; q < nreal; q++) { if (as_complex_real) cplx(shift); else real(); }
        if (as_complex_real && !only_complex) return;
        if (D == 4) cplx(1 + shift);
        cplx(1 + shift);
        cplx(2 + shift);
    };
    switch (tt) {
        case TT_SCALAR: real(); break;
        case TT_VEC3: real(); cplx(1); break;
        case TT_VEC4: real(); real(); cplx(1); break;
        case TT_SYM3: sym(3, 0, false, false); break;
        case TT_SYM4: sym(4, 0, false, false); break;
        default: {
            const int D1 = (tt == TT_R3_4_3 || tt == TT_R3_4_4) ? 4 : 3;
            const int D2 = (tt == TT_R3_3_4 || tt == TT_R3_4_4) ? 4 : 3;
            if (D1 == 4) sym(D2, 0, false, false);       // first index t
            sym(D2, 0, false, false);                     // first index r^
            sym(D2, 1, false, true);                      // [m; real entries]: complex, n = +1
            sym(D2, 1, true, false);                      // [m; complex entries]: n_e + 1
            sym(D2, -1, true, false);                     // [mbar; complex entries]: n_e - 1
        }
    }
}

template <bool INV>
static sp_status launch_pointwise(const std::vector<int> &types, const std::vector<TensorArgs> &targs, const std::vector<char> &sel,
                             const sp_shell *s, const double *src, double *dst, cudaStream_t st) {
    const int T = 128;
    const unsigned nb = (unsigned)(((size_t)s->Nr * s->Nt * (s->Nt + 1) + T - 1) / T);
    std::vector<char> done(types.size(), 0);
    const cudaStream_t main_st = st;
    bool forked = false;
    int nlaunch = 0;
    for (size_t t0 = 0; t0 < types.size(); t0++) {
        if (done[t0] || !sel[t0]) continue;
        // launches of different tensor groups are independent: every second one goes to the side stream
        if ((nlaunch++ & 1) && (forked || (forked = sp_fork(s, main_st)))) st = s->aux; else st = main_st;
        TensorArgsGroup tg;                      // this tensor and the following ones of the same index structure
        int n = 0;
        for (size_t t1 = t0; t1 < types.size() && n < SP_PW_GROUP; t1++)
            if (!done[t1] && sel[t1] && types[t1] == types[t0]) { tg.t[n++] = targs[t1]; done[t1] = 1; }
        const dim3 grid(nb, n);
#define SP_PW(TTV)                                                                                                        \
    case TTV:                                                                                                             \
        k_pointwise<TTV, INV><<<grid, T, 0, st>>>(tg, s->Nr, s->Nt, s->npts, s->d_sin_t, s->d_cos_t, s->d_sin_p, s->d_cos_p, \
                                                  src, dst);                                                              \
        break;
        switch (types[t0]) {
            SP_PW(TT_SCALAR) SP_PW(TT_VEC3) SP_PW(TT_VEC4) SP_PW(TT_SYM3) SP_PW(TT_SYM4) SP_PW(TT_R3_3_3) SP_PW(TT_R3_3_4)
            SP_PW(TT_R3_4_3) SP_PW(TT_R3_4_4)
        }
#undef SP_PW
        g_sp_launches += 1;
    }
    if (forked && !sp_join(s, main_st)) return SP_ERR_CUDA;      // an unjoined side stream would also invalidate a graph capture
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

// ---- fused filter stages (kernels_fused.cuh) --------------------------------------------------------------------------------
// Which tensors take the fused kernels.  Default (auto): tensors of up to 10 components (rank <= 2) whose data tiles leave three
// CTAs per SM and whose launch group fills at least two CTAs per SM -- where the fused kernels are as fast as the five-stage path on
// B200 and save its HBM round trips.  SP_FUSE = 0: never; 1: rank <= 2 whenever the tile fits; 2: every tensor
// whose tile fits (rank 3: analysis side only).
static int sp_fuse_mode() {
    static const int v = [] { const char *e = getenv("SP_FUSE"); return e ? atoi(e) : -1; }();
    return v;
}
static FusedParams fused_params(const sp_shell *s) {
    FusedParams fp;
    fp.Nr = s->Nr; fp.Nt = s->Nt; fp.L = s->L; fp.vec = s->Nr * s->Nt; fp.MC = s->MC;
    fp.npts = (long)s->npts; fp.dofsz = (long)s->MC4 * fp.vec;
    fp.sin_t = s->d_sin_t; fp.cos_t = s->d_cos_t; fp.sin_p = s->d_sin_p; fp.cos_p = s->d_cos_p;
    fp.Ac = s->d_fAc; fp.As = s->d_fAs; fp.Mp = s->f_Mp; fp.ldc = s->f_ldc; fp.lds = s->f_lds;
    fp.Sc = s->d_fSc; fp.Ss = s->d_fSs; fp.Jp = s->f_Jp; fp.ldk = s->f_ldk;
    fp.WM = 1; fp.WN = 1; fp.ngroup = 1; fp.nbuf = 1; fp.zs = 1;
    return fp;
}
// k_fan<TT, NC, MT, NTW, MAXT>: launch = true runs it, false only answers whether the tile fits
// tile buffers of the fused kernels: 1 (default: one work item per CTA, grid = item count) or, with SP_FUSE_NBUF = 2, two: a persistent
// grid whose CTAs stream the next item's tile in under the current item's products (measured slower on B200 at configs 2-5:
// the second buffer costs a resident CTA per SM)
static int fused_nbuf(size_t tile_bytes) {
    static const int forced = [] { const char *e = getenv("SP_FUSE_NBUF"); return e ? atoi(e) : 0; }();
    return (forced == 2 && 2 * tile_bytes <= (size_t)SP_SMEM_MAX) ? 2 : 1;
}
template <class K>
static sp_status fused_grid(K kernel, int nthr, size_t smem, int nitems, int nbuf, const sp_shell *s, int &grid) {
    grid = nitems;
    if (nbuf < 2) return SP_OK;
    int occ = 0;
    SP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, nthr, smem));
    if (occ < 1) return SP_ERR_CUDA;
    grid = std::min(nitems, occ * s->num_sms);
    return SP_OK;
}
template <int TT, int NC, int NTW, int MAXT>
static sp_status fan_launch(const sp_shell *s, const TensorArgsGroup &tg, int n, const double *src, double *coef, cudaStream_t st, bool launch,
                             size_t *tile_out, int *items_out) {
    constexpr int nc = TTInfo<TT>::nc, ntiles = nc * NC / 8, WN = (ntiles + NTW - 1) / NTW;
    static_assert(WN * 32 <= MAXT, "warp columns exceed the block size");
    const int mtiles = s->f_Mp / 8;
    const int MT = (nc > 10 || mtiles % 3 == 0 || mtiles >= 9) ? 3 : 2;
    const int WM = std::max(1, std::min(std::min(4, MAXT / 32 / WN), (mtiles + MT - 1) / MT));
    const size_t tile = fan_smem_bytes<NC>(nc, s->Np, 1);
    if (tile > (size_t)SP_SMEM_MAX) return SP_ERR_UNSUPPORTED;
    if (tile_out) *tile_out = tile;
    if (items_out) *items_out = ((s->Nr * s->Nt + NC - 1) / NC) * n;
    if (!launch) return SP_OK;
    FusedParams fp = fused_params(s);
    fp.WM = WM; fp.WN = WN; fp.ngroup = n; fp.nbuf = fused_nbuf(tile);
    const size_t smem = fan_smem_bytes<NC>(nc, s->Np, fp.nbuf);
    // further warps (up to SP_FAN_THREADS, default 128) only stage and project: the pointwise phase wants more threads than the products
    static const int minthr = [] { const char *e = getenv("SP_FAN_THREADS"); return e ? atoi(e) : 128; }();
    const int nthr = std::max(WM * WN * 32, std::min(MAXT, minthr));
    const int nitems = ((fp.vec + NC - 1) / NC) * n;
    int grid = 0;
    sp_status e;
    static bool attr3 = false, attr2 = false;
    if (MT == 3) {
        if (!attr3) { SP_CUDA(cudaFuncSetAttribute(k_fan<TT, NC, 3, NTW, MAXT>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX)); attr3 = true; }
        if ((e = fused_grid(k_fan<TT, NC, 3, NTW, MAXT>, nthr, smem, nitems, fp.nbuf, s, grid)) != SP_OK) return e;
        k_fan<TT, NC, 3, NTW, MAXT><<<grid, nthr, smem, st>>>(tg, fp, src, coef);
    } else {
        if (!attr2) { SP_CUDA(cudaFuncSetAttribute(k_fan<TT, NC, 2, NTW, MAXT>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX)); attr2 = true; }
        if ((e = fused_grid(k_fan<TT, NC, 2, NTW, MAXT>, nthr, smem, nitems, fp.nbuf, s, grid)) != SP_OK) return e;
        k_fan<TT, NC, 2, NTW, MAXT><<<grid, nthr, smem, st>>>(tg, fp, src, coef);
    }
    g_sp_launches += 1;
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}
static sp_status fan_dispatch(int tt, const sp_shell *s, const TensorArgsGroup &tg, int n, const double *src, double *coef, cudaStream_t st, bool launch,
                               size_t *tile_out = nullptr, int *items_out = nullptr) {
    // column tile and warp tiling per index structure: N = components x NC columns per CTA.  SP_FAN_NC4=1: 4-column tiles for the
    // symmetric rank-2 types (experiments)
    static const int nc4 = [] { const char *e = getenv("SP_FAN_NC4"); return e ? atoi(e) : 0; }();
    // small states: narrower column tiles, so that the launch has at least ~2 CTAs per SM
    const int vec = s->Nr * s->Nt;
    const bool narrow = (long)((vec + 63) / 64) * std::max(n, 1) < 2L * s->num_sms;
    const bool narrow16 = (long)((vec + 15) / 16) * std::max(n, 1) < 2L * s->num_sms;
    switch (tt) {
        case TT_SCALAR:
            if (narrow) return fan_launch<TT_SCALAR, 16, 2, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
            return fan_launch<TT_SCALAR, 64, 4, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
        case TT_VEC3:
            if (narrow16) return fan_launch<TT_VEC3, 8, 3, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
            return fan_launch<TT_VEC3, 16, 3, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
        case TT_VEC4:
            if (narrow16) return fan_launch<TT_VEC4, 8, 4, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
            return fan_launch<TT_VEC4, 16, 4, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
        case TT_SYM3: return fan_launch<TT_SYM3, 8, 3, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
        case TT_SYM4:
            if (nc4) return fan_launch<TT_SYM4, 4, 5, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
            return fan_launch<TT_SYM4, 8, 5, 512>(s, tg, n, src, coef, st, launch, tile_out, items_out);
        case TT_R3_3_3: return fan_launch<TT_R3_3_3, 4, 3, 256>(s, tg, n, src, coef, st, launch, tile_out, items_out);
        case TT_R3_3_4: return fan_launch<TT_R3_3_4, 4, 4, 256>(s, tg, n, src, coef, st, launch, tile_out, items_out);
        case TT_R3_4_3: return fan_launch<TT_R3_4_3, 4, 3, 256>(s, tg, n, src, coef, st, launch, tile_out, items_out);
        case TT_R3_4_4: return fan_launch<TT_R3_4_4, 4, 5, 256>(s, tg, n, src, coef, st, launch, tile_out, items_out);
    }
    return SP_ERR_UNSUPPORTED;
}
template <int TT, int CBW>
static sp_status fsyn_launch(const sp_shell *s, const TensorArgsGroup &tg, int n, const double *coef, double *dst, cudaStream_t st, bool launch,
                              size_t *tile_out, int *items_out) {
    constexpr int nc = TTInfo<TT>::nc, NC = 8 * CBW;
    // at most SP_FSYN_NW (default 4) warps per CTA: more CTAs along the longitudes share a column tile when there are more 8-row tiles
    static const int nwmax = [] { const char *e = getenv("SP_FSYN_NW"); const int v = e ? atoi(e) : 4; return v >= 1 && v <= 8 ? v : 4; }();
    const int jtiles = s->f_Jp / 8, zs = (jtiles + nwmax - 1) / nwmax, nw = (jtiles + zs - 1) / zs;
    const size_t tile = fsyn_smem_bytes(nc, s->MC, NC, 1);
    if (tile > (size_t)SP_SMEM_MAX) return SP_ERR_UNSUPPORTED;
    if (tile_out) *tile_out = tile;
    if (items_out) *items_out = ((s->Nr * s->Nt + NC - 1) / NC) * zs * n;
    if (!launch) return SP_OK;
    FusedParams fp = fused_params(s);
    fp.ngroup = n; fp.zs = zs; fp.nbuf = fused_nbuf(tile);
    const size_t smem = fsyn_smem_bytes(nc, s->MC, NC, fp.nbuf);
    static bool attr = false;
    if (!attr) { SP_CUDA(cudaFuncSetAttribute(k_fsyn<TT, CBW>, cudaFuncAttributeMaxDynamicSharedMemorySize, SP_SMEM_MAX)); attr = true; }
    const int nitems = ((fp.vec + NC - 1) / NC) * zs * n;
    int grid = 0;
    sp_status e = fused_grid(k_fsyn<TT, CBW>, nw * 32, smem, nitems, fp.nbuf, s, grid);
    if (e != SP_OK) return e;
    k_fsyn<TT, CBW><<<grid, nw * 32, smem, st>>>(tg, fp, coef, dst);
    g_sp_launches += 1;
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}
static sp_status fsyn_dispatch(int tt, const sp_shell *s, const TensorArgsGroup &tg, int n, const double *coef, double *dst, cudaStream_t st, bool launch,
                                size_t *tile_out = nullptr, int *items_out = nullptr) {
    const int vec = s->Nr * s->Nt;
    const bool narrow = (long)((vec + 63) / 64) * std::max(n, 1) < 2L * s->num_sms;
    const bool narrow16 = (long)((vec + 15) / 16) * std::max(n, 1) < 2L * s->num_sms;
    switch (tt) {
        case TT_SCALAR:
            if (narrow) return fsyn_launch<TT_SCALAR, 2>(s, tg, n, coef, dst, st, launch, tile_out, items_out);
            return fsyn_launch<TT_SCALAR, 8>(s, tg, n, coef, dst, st, launch, tile_out, items_out);
        case TT_VEC3:
            if (narrow16) return fsyn_launch<TT_VEC3, 1>(s, tg, n, coef, dst, st, launch, tile_out, items_out);
            return fsyn_launch<TT_VEC3, 2>(s, tg, n, coef, dst, st, launch, tile_out, items_out);
        case TT_VEC4:
            if (narrow16) return fsyn_launch<TT_VEC4, 1>(s, tg, n, coef, dst, st, launch, tile_out, items_out);
            return fsyn_launch<TT_VEC4, 2>(s, tg, n, coef, dst, st, launch, tile_out, items_out);
        case TT_SYM3: return fsyn_launch<TT_SYM3, 1>(s, tg, n, coef, dst, st, launch, tile_out, items_out);
        case TT_SYM4: return fsyn_launch<TT_SYM4, 1>(s, tg, n, coef, dst, st, launch, tile_out, items_out);
    }
    return SP_ERR_UNSUPPORTED;      // rank 3: the lane-local recombination would need > 255 registers; five-stage path
}
// joins the shell's side stream back into the caller's stream on every exit path (a fork left open would invalidate a CUDA
// graph capture and hide the original error)
struct AuxJoin {
    const sp_shell *s; cudaStream_t st; bool open = false;
    bool fork() { if (!open) open = sp_fork(s, st); return open; }
    bool join() { if (!open) return true; open = false; return sp_join(s, st); }
    ~AuxJoin() { if (open) sp_join(s, st); }
};

// run `fn(type, group, count, stream)` over the selected tensors, grouped by index structure (up to SP_PW_GROUP tensors per launch);
// the launches of different groups are independent: every second one goes to the shell's side stream
template <class Fn, class Aux>
static sp_status for_groups(const std::vector<int> &types, const std::vector<TensorArgs> &targs, const std::vector<char> &sel,
                            cudaStream_t st, Aux &aux, Fn fn) {
    std::vector<char> done(types.size(), 0);
    int nlaunch = 0;
    for (size_t t0 = 0; t0 < types.size(); t0++) {
        if (done[t0] || !sel[t0]) continue;
        TensorArgsGroup tg;
        int n = 0;
        for (size_t t1 = t0; t1 < types.size() && n < SP_PW_GROUP; t1++)
            if (!done[t1] && sel[t1] && types[t1] == types[t0]) { tg.t[n++] = targs[t1]; done[t1] = 1; }
        const cudaStream_t sx = ((nlaunch++ & 1) && aux.fork()) ? aux.s->aux : st;
        sp_status e = fn(types[t0], tg, n, sx);
        if (e != SP_OK) return e;
    }
    return SP_OK;
}

extern "C" sp_status sp_tensor_filter(const sp_shell *s, const double *u, double *out, int nfields, const sp_tensor_desc *tens,
                                      int ntens, void *ws, size_t wsb, void *stream) {
    if (!s || !u || !out || nfields < 0 || ntens < 0 || (ntens > 0 && !tens)) return SP_ERR_INVALID_ARG;
    if (!s->built) return SP_ERR_NOT_BUILT;
    cudaStream_t st = (cudaStream_t)stream;
    const int Nr = s->Nr, Nt = s->Nt;
    const size_t npts = s->npts, vec = (size_t)Nt * Nr;
    // ---- validate, classify, build the component list
    std::vector<int> owner(nfields, -1), types(ntens);
    std::vector<TensorArgs> targs(ntens);
    std::vector<ThetaComp> comps;
    int ndof = 0;
    for (int t = 0; t < ntens; t++) {
        const sp_tensor_desc &d = tens[t];
        if (d.rank < 0 || d.rank > 3 || !d.field) return SP_ERR_INVALID_ARG;
        int tt = classify(d);
        if (tt == -1) return SP_ERR_INVALID_ARG;
        if (tt < 0) return SP_ERR_UNSUPPORTED;
        types[t] = tt;
        TensorArgs &a = targs[t];
        a.ncomp = tt_ncomp(tt);
        a.dof0 = ndof;
        for (int c = 0; c < a.ncomp; c++) {
            int f = d.field[c];
            if (f < 0 || f >= nfields || owner[f] >= 0) return SP_ERR_INVALID_ARG;
            owner[f] = t;
            a.field[c] = f;
        }
        tt_components(tt, ndof, comps);
        ndof += a.ncomp;
    }
    if (out != u)
        for (int f = 0; f < nfields; f++)
            if (owner[f] < 0) SP_CUDA(cudaMemcpyAsync(out + f * npts, u + f * npts, npts * sizeof(double), cudaMemcpyDeviceToDevice, st));
    if (ndof == 0) return SP_OK;
    const size_t need = (size_t)ndof * (npts + 2 * (size_t)s->MC4 * vec) * sizeof(double);
    if (!ws || wsb < need) return SP_ERR_INVALID_ARG;
    double *dofs = (double *)ws, *coef1 = dofs + (size_t)ndof * npts, *coef2 = coef1 + (size_t)ndof * s->MC4 * vec;
    // ---- which tensors take the fused kernels (F1+F2 in k_fan, F4+F5 in k_fsyn): 16-byte aligned buffers, even strides, tile fits
    std::vector<char> fanF(ntens, 0), synF(ntens, 0), fanU(ntens, 1), synU(ntens, 1);
    const int fmode = sp_fuse_mode();
    const bool fusable = fmode != 0 && s->d_fAc && !(vec & 1) && !(((uintptr_t)u | (uintptr_t)out | (uintptr_t)ws) & 15);
    bool anyFanU = false, anySynU = false;
    for (int t = 0; t < ntens; t++) {
        if (fusable && (fmode > 1 || targs[t].ncomp <= 10)) {
            TensorArgsGroup none;
            int nsame = 0;                                   // tensors of this index structure: they share a launch
            for (int q = 0; q < ntens; q++) nsame += types[q] == types[t];
            nsame = std::min(nsame, SP_PW_GROUP);
            size_t tf = 0, ts = 0;
            int itf = 0, its = 0;
            fanF[t] = fan_dispatch(types[t], s, none, nsame, nullptr, nullptr, st, false, &tf, &itf) == SP_OK;
            synF[t] = fsyn_dispatch(types[t], s, none, nsame, nullptr, nullptr, st, false, &ts, &its) == SP_OK;
            if (fmode < 0) {                                 // auto: both sides, three CTAs per SM, two CTAs per SM in flight
                const size_t lim = (size_t)SP_SMEM_MAX / 3 - 1024;
                const bool ok = fanF[t] && synF[t] && tf <= lim && ts <= lim && itf >= 2 * s->num_sms && its >= 2 * s->num_sms;
                fanF[t] = synF[t] = ok;
            }
        }
        fanU[t] = !fanF[t]; synU[t] = !synF[t];
        anyFanU |= fanU[t] != 0; anySynU |= synU[t] != 0;
    }
    // contiguous dof ranges of the tensors that take the five-stage path (the phi products run per range)
    auto ranges = [&](const std::vector<char> &sel) {
        std::vector<std::pair<int, int>> r;
        for (int t = 0; t < ntens; t++) {
            if (!sel[t]) continue;
            if (!r.empty() && r.back().first + r.back().second == targs[t].dof0) r.back().second += targs[t].ncomp;
            else r.push_back({targs[t].dof0, targs[t].ncomp});
        }
        return r;
    };
    AuxJoin aux{s, st};
    const long cst = (long)(s->MC4 * vec);
    auto phi = [&](const sp_shell::PhiMat &pm, const double *B, long sBb, double *C, long sCb, int nb, cudaStream_t sx) -> sp_status {
        if (pm.M <= 0 || pm.K <= 0) return SP_OK;
        PhiTiling tl = {pm.MT, pm.mg, pm.Mpad};
        sp_status e = launch_phi_gemm(pm.d, pm.K8, pm.M, tl, pm.K, B, (long)vec, sBb, C, (long)vec, sCb, (int)vec, nb, sx, s->num_sms);
        if (e == SP_ERR_UNSUPPORTED)      // odd strides: generic global-memory kernel (same padded matrix)
            e = launch_gemm_cols<false>(pm.d, pm.K8, pm.M, pm.K, B, (long)vec, sBb, C, (long)vec, sCb, (int)vec, nb, sx);
        g_sp_launches += 1;
        return e;
    };
    sp_status e;
    // ---- F1: dyad projection (five-stage tensors)
    sp_mark(s, st, 3);
    if (anyFanU && (e = launch_pointwise<false>(types, targs, fanU, s, u, dofs, st)) != SP_OK) return e;
    sp_mark(s, st, 4);
    // ---- F1 + F2 fused; F2: phi analysis (eq. 33) on the folded rows: cosine block -> a_0..a_L, sine block -> b_1..b_L
    e = for_groups(types, targs, fanF, st, aux, [&](int tt, const TensorArgsGroup &tg, int n, cudaStream_t sx) { return fan_dispatch(tt, s, tg, n, u, coef1, sx, true); });
    if (e != SP_OK) return e;
    if (anyFanU) {
        // the cosine and the sine block are independent: the sine block runs on the side stream
        const bool fk = s->m_as.M > 0 && s->m_as.K > 0 && aux.fork();
        for (const auto &r : ranges(fanU)) {
            const double *B = dofs + (size_t)r.first * npts;
            double *C = coef1 + (size_t)r.first * cst;
            if ((e = phi(s->m_ac, B, (long)npts, C, cst, r.second, st)) != SP_OK) return e;
            if ((e = phi(s->m_as, B + (size_t)(Nt + 1) * vec, (long)npts, C + (size_t)(s->L + 1) * vec, cst, r.second, fk ? s->aux : st)) != SP_OK) return e;
        }
    }
    if (!aux.join()) return SP_ERR_CUDA;      // fused launches on the side stream and the sine blocks are back before the theta step
    sp_mark(s, st, 5);
    // ---- F3: per-(n,m) theta matrices (eq. 62)
    {
        const int mtiles = s->Nt8 / 8;
        if (s->theta_NT > 0) {
            std::vector<ThetaComp2> rl, cx;
            for (const ThetaComp &c : comps) (c.cplx ? cx : rl).push_back({c.dof, c.n});
            sp_status e2 = launch_theta2(s, s->theta_NT, rl, cx, coef1, coef2, st);
            if (e2 != SP_OK) return e2;
        } else {   // very large Ntheta: generic global-memory kernel
            const int nwarps = (Nr + 3) / 4;
            if (nwarps > 20) return SP_ERR_UNSUPPORTED;
            for (size_t c0 = 0; c0 < comps.size(); c0 += SP_THETA_BATCH) {
                ThetaBatch b;
                int nb = (int)std::min<size_t>(SP_THETA_BATCH, comps.size() - c0);
                for (int q = 0; q < nb; q++) b.c[q] = comps[c0 + q];
                dim3 grid(s->L + 1, nb, (mtiles + 3) / 4);
                k_theta<4><<<grid, nwarps * 32, 0, st>>>(b, s->d_F, s->L, Nt, s->Nt8, s->Nt8, Nr, s->MC4, coef1, coef2);
                g_sp_launches += 1;
            }
        }
        if (cudaGetLastError() != cudaSuccess) return SP_ERR_CUDA;
    }
    sp_mark(s, st, 6);
    // ---- F4 + F5 fused; F4: phi synthesis (eq. 31) into the folded rows: e_j (cosine block), o_j (sine block)
    e = for_groups(types, targs, synF, st, aux, [&](int tt, const TensorArgsGroup &tg, int n, cudaStream_t sx) { return fsyn_dispatch(tt, s, tg, n, coef2, out, sx, true); });
    if (e != SP_OK) return e;
    if (anySynU) {
        const bool fk = s->m_ss.M > 0 && s->m_ss.K > 0 && aux.fork();
        for (const auto &r : ranges(synU)) {
            const double *C = coef2 + (size_t)r.first * cst;
            double *B = dofs + (size_t)r.first * npts;
            if ((e = phi(s->m_sc, C, cst, B, (long)npts, r.second, st)) != SP_OK) return e;
            if ((e = phi(s->m_ss, C + (size_t)(s->L + 1) * vec, cst, B + (size_t)(Nt + 1) * vec, (long)npts, r.second, fk ? s->aux : st)) != SP_OK) return e;
            if (s->m_ss.K <= 0 && Nt > 1)      // L = 0: no sine modes survive, the odd rows o_j are zero
                SP_CUDA(cudaMemset2DAsync(B + (size_t)(Nt + 1) * vec, npts * sizeof(double), 0, (size_t)(Nt - 1) * vec * sizeof(double),
                                          (size_t)r.second, st));
        }
    }
    if (!aux.join()) return SP_ERR_CUDA;
    sp_mark(s, st, 7);
    // ---- F5: recombination (five-stage tensors)
    if (anySynU && (e = launch_pointwise<true>(types, targs, synU, s, dofs, out, st)) != SP_OK) return e;
    sp_mark(s, st, 8);
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

extern "C" sp_status sp_rhs_wave_shell(const sp_shell *s, const double *u, double *dudt, int bc_inner, int bc_outer, void *ws, size_t wsb,
                                       void *stream) {
    if (!s || !u || !dudt) return SP_ERR_INVALID_ARG;
    if (!s->built) return SP_ERR_NOT_BUILT;
    const size_t npts = s->npts;
    if (!ws || wsb < 16 * npts * sizeof(double)) return SP_ERR_INVALID_ARG;
    double *gws = (double *)ws, *dg = gws + 4 * npts;
    sp_status e = sp_cartesian_gradient(s, u + npts, 4, dg, gws, 4 * npts * sizeof(double), stream);
    if (e != SP_OK) return e;
    const int T = 256;
    g_sp_launches += 1;
    k_wave_rhs<<<(unsigned)((npts + T - 1) / T), T, 0, (cudaStream_t)stream>>>(s->Nr, s->Nt, npts, s->d_sin_t, s->d_cos_t, s->d_sin_p,
                                                                              s->d_cos_p, u, dg, dudt, (bc_inner ? 1 : 0) | (bc_outer ? 2 : 0));
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

extern "C" sp_status sp_rhs_first_order_wave(const sp_shell *s, const double *u, double *dudt, void *ws, size_t wsb, void *stream) {
    return sp_rhs_wave_shell(s, u, dudt, 1, 1, ws, wsb, stream);
}

extern "C" sp_status sp_wave_interface(const sp_shell *a, double *da, const sp_shell *b, double *db, void *stream) {
    if (!a || !b || !da || !db || a == b) return SP_ERR_INVALID_ARG;
    if (!a->built || !b->built) return SP_ERR_NOT_BUILT;
    if (a->Nt != b->Nt || a->Np != b->Np || fabs(a->rout - b->rin) > 1e-12 * fabs(a->rout)) return SP_ERR_INVALID_ARG;
    const int n = a->Nt * a->Np;
    g_sp_launches += 1;
    k_wave_interface<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(a->Nt, a->Np, a->Nr, b->Nr, a->d_sin_t, a->d_cos_t, a->d_sin_p,
                                                                      a->d_cos_p, da, db);
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

// ---- GHG system (Appendix A)
extern "C" sp_status sp_ghg_workspace_bytes(const sp_shell *s, size_t *bytes) {
    if (!s || !bytes) return SP_ERR_INVALID_ARG;
    *bytes = (size_t)(150 + 50) * s->npts * sizeof(double);      // gradient of the 50 fields + the gradient call's own workspace
    return SP_OK;
}

extern "C" sp_status sp_rhs_ghg(const sp_shell *s, const double *u, const double *H, const double *dH, double *dudt, int bc_outer,
                                void *ws, size_t wsb, void *stream) {
    if (!s || !u || !H || !dH || !dudt || dudt == u) return SP_ERR_INVALID_ARG;
    if (!s->built) return SP_ERR_NOT_BUILT;
    const size_t npts = s->npts;
    if (!ws || wsb < 200 * npts * sizeof(double)) return SP_ERR_INVALID_ARG;
    double *du = (double *)ws, *gws = du + 150 * npts;
    sp_status e = sp_cartesian_gradient(s, u, 50, du, gws, 50 * npts * sizeof(double), stream);
    if (e != SP_OK) return e;
    GhgArgs A = {u, du, H, dH, dudt, npts};
    g_sp_launches += 1;
    k_ghg_rhs<<<(unsigned)((npts + 127) / 128), 128, 0, (cudaStream_t)stream>>>(A);
    if (bc_outer) {
        const int nb = s->Nt * s->Np;
        g_sp_launches += 1;
        k_ghg_bc<<<(nb + 127) / 128, 128, 0, (cudaStream_t)stream>>>(u, dudt, npts, s->Nr, s->Nt, s->Np, s->d_sin_t, s->d_cos_t, s->d_sin_p,
                                                                      s->d_cos_p);
    }
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

extern "C" sp_status sp_ghg_init(const sp_shell *s, double *u, double *H, void *stream) {
    if (!s || !u || !H) return SP_ERR_INVALID_ARG;
    if (!s->built) return SP_ERR_NOT_BUILT;
    g_sp_launches += 1;
    k_ghg_init<<<(unsigned)((s->npts + 127) / 128), 128, 0, (cudaStream_t)stream>>>(u, H, s->npts);
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

extern "C" sp_status sp_wave_dt(const sp_shell *s, double lambda, double *dt) {
    if (!s || !dt || !(lambda > 0)) return SP_ERR_INVALID_ARG;
    const double PI = 3.14159265358979323846;
    const double mid = 0.5 * (s->rout + s->rin), half = 0.5 * (s->rout - s->rin);
    const double r0 = mid - half, r1 = mid - half * cos(PI / (s->Nr - 1));                 // eq. 2
    const double th0 = PI * 0.5 / s->Nt;                                                   // eq. 3
    const double dphi = 2.0 * r0 * sin(th0) * sin(PI / s->Np);
    *dt = lambda * std::min(r1 - r0, dphi);                                                // eq. 63
    return SP_OK;
}

extern "C" sp_status sp_ghg_graded_degree(const sp_shell *s, int field, int *L_out) {
    if (!s || !L_out || field < 0 || field >= 50) return SP_ERR_INVALID_ARG;
    static const int ab[10] = {0, 1, 1, 1, 2, 2, 2, 2, 2, 2};            // tt, tx, ty, tz, xx, xy, xz, yy, yz, zz
    const int d = ab[field % 10] + (field >= 20 ? 1 : 0);                 // d_iab carries one more spatial index
    *L_out = std::min(s->L + d, s->Nt - 1);
    return SP_OK;
}

extern "C" sp_status sp_axpby(double a, const double *x, double b, double *y, size_t n, void *stream) {
    if (!x || !y) return SP_ERR_INVALID_ARG;
    if (n == 0) return SP_OK;
    size_t nb = (n + 255) / 256;
    if (nb > 148 * 16) nb = 148 * 16;
    g_sp_launches += 1;
    k_axpby<<<(unsigned)nb, 256, 0, (cudaStream_t)stream>>>(a, x, b, y, n);
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

extern "C" sp_status sp_rk4_stage(const double *u, const double *k, const double *acc_in, double *acc_out, double *stage_out,
                                  double c_acc, double c_stage, size_t n, void *stream) {
    if (!u || !k || !acc_in || !acc_out) return SP_ERR_INVALID_ARG;
    if (stage_out == u || stage_out == k || stage_out == acc_in || (stage_out && stage_out == acc_out) || acc_out == k)
        return SP_ERR_INVALID_ARG;
    if (n == 0) return SP_OK;
    size_t nb = (n + 255) / 256;
    if (nb > 148 * 16) nb = 148 * 16;
    g_sp_launches += 1;
    k_rk4_stage<<<(unsigned)nb, 256, 0, (cudaStream_t)stream>>>(u, k, acc_in, acc_out, stage_out, c_acc, c_stage, n);
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}

extern "C" sp_status sp_probe_fp64_peak(int mode, double *tflops) {
    if (!tflops || mode < 0 || mode > 1) return SP_ERR_INVALID_ARG;
    cudaDeviceProp prop;
    int dev = 0;
    SP_CUDA(cudaGetDevice(&dev));
    SP_CUDA(cudaGetDeviceProperties(&prop, dev));
    const int grid = prop.multiProcessorCount * 2, thr = 512, iters = 20000;
    double *buf = nullptr;
    SP_CUDA(cudaMalloc((void **)&buf, sizeof(double) * grid * thr));
    cudaEvent_t e0, e1;
    SP_CUDA(cudaEventCreate(&e0));
    SP_CUDA(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 6; rep++) {
        cudaEventRecord(e0);
        if (mode == 0) k_probe_dmma<<<grid, thr>>>(buf, iters, 1.0000001, 1e-9);
        else k_probe_dfma<<<grid, thr>>>(buf, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(buf); return SP_ERR_CUDA; }
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    const double flops = (mode == 0) ? 2.0 * 256 * 8 * iters * (double)grid * (thr / 32) : 2.0 * 16 * iters * (double)grid * thr;
    *tflops = flops / (best * 1e-3) * 1e-12;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf);
    return SP_OK;
}

extern "C" sp_status sp_profile_enable(sp_shell *s, int on) {
    if (!s) return SP_ERR_INVALID_ARG;
    if (on)
        for (int q = 0; q < 9; q++)
            if (!s->ev[q]) SP_CUDA(cudaEventCreate(&s->ev[q]));
    for (int q = 0; q < 9; q++) s->ev_set[q] = false;
    s->prof = on != 0;
    return SP_OK;
}

extern "C" sp_status sp_profile_read(const sp_shell *s, double *ms7) {
    if (!s || !ms7) return SP_ERR_INVALID_ARG;
    int a[7] = {0, 1, 3, 4, 5, 6, 7}, b[7] = {1, 2, 4, 5, 6, 7, 8};
    if (s->grad_swapped) { a[0] = 1; b[0] = 2; a[1] = 0; b[1] = 1; }      // (r,theta) kernel ran first
    for (int q = 0; q < 7; q++) {
        ms7[q] = -1.0;
        if (s->ev_set[a[q]] && s->ev_set[b[q]]) {
            SP_CUDA(cudaEventSynchronize(s->ev[b[q]]));
            float ms = 0;
            SP_CUDA(cudaEventElapsedTime(&ms, s->ev[a[q]], s->ev[b[q]]));
            ms7[q] = ms;
        }
    }
    return SP_OK;
}

extern "C" unsigned long long sp_launch_count(void) { return g_sp_launches; }

// =================================================================================================
// sp_tensor_filter_noalloc: the Yn filter with its scratch in a file-scope static device array (spshell.h).
// In HOST code `g_sp_noalloc_scratch` is only a stand-in for the symbol, not a device address: the device address is resolved
// once per device with cudaGetSymbolAddress (that device current) and that pointer is what the kernels get.
// =================================================================================================
static __device__ __align__(256) unsigned char g_sp_noalloc_scratch[SP_NOALLOC_SCRATCH_BYTES];

#include <mutex>
static const int SP_NOALLOC_MAXDEV = 64;
static void *g_sp_noalloc_ptr[SP_NOALLOC_MAXDEV] = {};      // device address of the array on device d (null: not resolved yet)
static std::mutex g_sp_noalloc_mu;

static sp_status sp_noalloc_scratch(void **out) {
    int dev = -1;
    SP_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= SP_NOALLOC_MAXDEV) return SP_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_sp_noalloc_mu);
    if (!g_sp_noalloc_ptr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_sp_noalloc_scratch) != cudaSuccess || !p) return SP_ERR_CUDA;
        g_sp_noalloc_ptr[dev] = p;
    }
    *out = g_sp_noalloc_ptr[dev];
    return SP_OK;
}

extern "C" sp_status sp_tensor_filter_noalloc(const sp_shell *s, const double *u, double *out, int nfields, const sp_tensor_desc *tens,
                                              int ntens, void *stream) {
    if (!s || !u || !out || nfields < 0 || ntens < 0 || (ntens > 0 && !tens)) return SP_ERR_INVALID_ARG;
    if (!s->built) return SP_ERR_NOT_BUILT;
    // scratch the call needs (as sp_tensor_filter computes it); malformed descriptors are left to sp_tensor_filter's own checks
    size_t ndof = 0;
    for (int t = 0; t < ntens; t++) {
        if (tens[t].rank < 0 || tens[t].rank > 3 || !tens[t].field) return SP_ERR_INVALID_ARG;
        const int tt = classify(tens[t]);
        if (tt == -1) return SP_ERR_INVALID_ARG;
        if (tt < 0) return SP_ERR_UNSUPPORTED;
        ndof += (size_t)tt_ncomp(tt);
    }
    const size_t vec = (size_t)s->Nt * s->Nr;
    const size_t need = ndof * (s->npts + 2 * (size_t)s->MC4 * vec) * sizeof(double);
    if (need > (size_t)SP_NOALLOC_SCRATCH_BYTES) return SP_ERR_SCRATCH_LIMIT;      // nothing launched
    void *ws = nullptr;
    const sp_status e = sp_noalloc_scratch(&ws);
    if (e != SP_OK) return e;
    return sp_tensor_filter(s, u, out, nfields, tens, ntens, ws, (size_t)SP_NOALLOC_SCRATCH_BYTES, stream);
}
