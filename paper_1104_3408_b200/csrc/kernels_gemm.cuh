// Batched "small matrix x wide strided slab" FP64 contraction on the DMMA tensor path:
//     C[b][m][c] = sum_k A[m][k] * B[b][k][c],   m < M, k < K, c < ncols,
// B[b][k][c] = B + b*sBb + k*sBk + c (columns contiguous), C likewise with sCm, sCb.
// This is the paper's product (18) / (33) / (31) WITHOUT the transposes (17), (19):
// the contraction index has the large stride, the column index is contiguous.
//   CIRC = true : A[m][k] = g[(m - k) mod n]  (Fourier differentiation matrix, eq. 8, circulant), lda = n
//   CIRC = false: A row-major [rows padded to 8][lda], zero padded, lda >= K rounded up to 4
// One warp owns MT m-tiles x NT n-tiles (8x8 each) and walks K in steps of 4.
#pragma once
#include "sp_device.cuh"

template <int MT, int NT, bool CIRC>
__global__ void __launch_bounds__(256)
k_gemm_cols(const double *__restrict__ A, int lda, int M, int K, const double *__restrict__ B, long sBk, long sBb,
            double *__restrict__ C, long sCm, long sCb, int ncols) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const int nt0 = (blockIdx.x * (blockDim.x >> 5) + warp) * NT;
    if (nt0 * 8 >= ncols) return;
    const int mt0 = blockIdx.z * MT;
    const double *Bb = B + (long)blockIdx.y * sBb;
    double *Cb = C + (long)blockIdx.y * sCb;

    double acc[MT][NT][2];
#pragma unroll
    for (int a = 0; a < MT; a++)
#pragma unroll
        for (int b = 0; b < NT; b++) acc[a][b][0] = acc[a][b][1] = 0.0;

    int col[NT];
    bool cok[NT];
#pragma unroll
    for (int b = 0; b < NT; b++) {
        col[b] = (nt0 + b) * 8 + g;
        cok[b] = col[b] < ncols;
    }
    const int ksteps = (K + 3) >> 2;
#pragma unroll 2
    for (int ks = 0; ks < ksteps; ks++) {
        const int k = ks * 4 + t;
        const bool kok = k < K;
        double bf[NT], af[MT];
#pragma unroll
        for (int b = 0; b < NT; b++) bf[b] = (kok && cok[b]) ? __ldg(Bb + (long)k * sBk + col[b]) : 0.0;
#pragma unroll
        for (int a = 0; a < MT; a++) {
            const int row = (mt0 + a) * 8 + g;
            if (CIRC) {
                int d = row - k;
                d += (d < 0) ? lda : 0;
                af[a] = (row < M && kok) ? __ldg(A + d) : 0.0;
            } else {
                af[a] = (row < M && kok) ? __ldg(A + (long)row * lda + k) : 0.0;
            }
        }
#pragma unroll
        for (int a = 0; a < MT; a++)
#pragma unroll
            for (int b = 0; b < NT; b++) dmma(acc[a][b][0], acc[a][b][1], af[a], bf[b]);
    }
#pragma unroll
    for (int a = 0; a < MT; a++) {
        const int row = (mt0 + a) * 8 + g;
        if (row >= M) continue;
#pragma unroll
        for (int b = 0; b < NT; b++) {
            const int c0 = (nt0 + b) * 8 + 2 * t;
            double *p = Cb + (long)row * sCm + c0;
            if (c0 < ncols) p[0] = acc[a][b][0];
            if (c0 + 1 < ncols) p[1] = acc[a][b][1];
        }
    }
}

// Host launcher: picks MT so that blockIdx.z covers all m-tiles.
template <bool CIRC>
static sp_status launch_gemm_cols(const double *A, int lda, int M, int K, const double *B, long sBk, long sBb, double *C,
                                  long sCm, long sCb, int ncols, int nbatch, cudaStream_t st) {
    const int mtiles = (M + 7) / 8, ntiles = (ncols + 7) / 8;
    constexpr int NT = 2, WARPS = 8;
    dim3 block(WARPS * 32);
    const int nx = (ntiles + NT * WARPS - 1) / (NT * WARPS);
    if (mtiles % 6 == 0 || mtiles > 8) {
        dim3 grid(nx, nbatch, (mtiles + 5) / 6);
        k_gemm_cols<6, NT, CIRC><<<grid, block, 0, st>>>(A, lda, M, K, B, sBk, sBb, C, sCm, sCb, ncols);
    } else if (mtiles > 4) {
        dim3 grid(nx, nbatch, (mtiles + 3) / 4);
        k_gemm_cols<4, NT, CIRC><<<grid, block, 0, st>>>(A, lda, M, K, B, sBk, sBb, C, sCm, sCb, ncols);
    } else if (mtiles > 2) {
        dim3 grid(nx, nbatch, (mtiles + 3) / 4);
        k_gemm_cols<4, NT, CIRC><<<grid, block, 0, st>>>(A, lda, M, K, B, sBk, sBb, C, sCm, sCb, ncols);
    } else {
        dim3 grid(nx, nbatch, (mtiles + 1) / 2);
        k_gemm_cols<2, NT, CIRC><<<grid, block, 0, st>>>(A, lda, M, K, B, sBk, sBb, C, sCm, sCb, ncols);
    }
    return cudaGetLastError() == cudaSuccess ? SP_OK : SP_ERR_CUDA;
}
