// S3: dense FP64 building blocks for the port-level system ("one decomposition",
// PAPER.md:202 substitution for the m+n right-hand sides): generic-stride GEMM, blocked Cholesky,
// blocked forward triangular solve (used to invert the diagonal Cholesky factors).  All matrices row-major with a leading
// dimension; every kernel is bounds-checked (arbitrary sizes).
#pragma once
#include "common.cuh"

namespace pdn {

constexpr int GEMM_BM = 64, GEMM_BN = 64, GEMM_BK = 16;
constexpr int DENSE_NB = 32;  // panel width of the blocked factor / solves

// C[i*ldc + j] = beta * C + alpha * sum_k A(i,k) B(k,j),  A(i,k) = A[i*sai + k*sak], B(k,j) = B[k*sbk + j*sbj].
// 256 threads, 64x64 tile, 4x4 register tile per thread.
__global__ void __launch_bounds__(256)
k_gemm(int M, int N, int K, double alpha, const double* __restrict__ A, int64_t sai, int64_t sak,
       const double* __restrict__ B, int64_t sbk, int64_t sbj, double beta, double* __restrict__ C, int64_t ldc) {
    __shared__ double As[GEMM_BK][GEMM_BM + 1];
    __shared__ double Bs[GEMM_BK][GEMM_BN + 1];
    const int tid = threadIdx.x;
    const int tx = tid % 16, ty = tid / 16;
    const int i0 = blockIdx.y * GEMM_BM, j0 = blockIdx.x * GEMM_BN;
    double acc[4][4] = {};
    for (int k0 = 0; k0 < K; k0 += GEMM_BK) {
        for (int e = tid; e < GEMM_BK * GEMM_BM; e += 256) {
            // choose the fastest-varying index to follow the unit stride of the operand
            int kk, ii;
            if (sak == 1) { kk = e % GEMM_BK; ii = e / GEMM_BK; } else { ii = e % GEMM_BM; kk = e / GEMM_BM; }
            const int gi = i0 + ii, gk = k0 + kk;
            As[kk][ii] = (gi < M && gk < K) ? A[gi * sai + gk * sak] : 0.0;
        }
        for (int e = tid; e < GEMM_BK * GEMM_BN; e += 256) {
            int kk, jj;
            if (sbk == 1) { kk = e % GEMM_BK; jj = e / GEMM_BK; } else { jj = e % GEMM_BN; kk = e / GEMM_BN; }
            const int gj = j0 + jj, gk = k0 + kk;
            Bs[kk][jj] = (gj < N && gk < K) ? B[gk * sbk + gj * sbj] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < GEMM_BK; ++kk) {
            double a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) a[r] = As[kk][ty * 4 + r];
#pragma unroll
            for (int c = 0; c < 4; ++c) b[c] = Bs[kk][tx + 16 * c];
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[r][c] = fma(a[r], b[c], acc[r][c]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int gi = i0 + ty * 4 + r;
        if (gi >= M) continue;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int gj = j0 + tx + 16 * c;
            if (gj >= N) continue;
            double* p = C + gi * ldc + gj;
            *p = (beta == 0.0) ? alpha * acc[r][c] : fma(alpha, acc[r][c], beta * *p);
        }
    }
}

// Same contraction on the FP64 tensor cores (DMMA, mma.sync m8n8k4): 128x128 block tile, 8 warps in a 2x4
// grid, each accumulating a 64x32 tile as 8x4 m8n8 fragments; K is walked in steps of 16 through shared memory
// (k-major tiles padded by 8 so that the four k-rows of a fragment load fall in two conflict-free wavefronts),
// the next tile's global loads overlapping the current tile's MMAs in registers.  Any strides, any sizes.
constexpr int DG_BM = 128, DG_BN = 128, DG_BK = 16, DG_PAD = 8, DG_THREADS = 256;

__device__ __forceinline__ void dmma_m8n8k4(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(DG_THREADS)
k_gemm_dmma(int M, int N, int K, double alpha, const double* __restrict__ A, int64_t sai, int64_t sak,
            const double* __restrict__ B, int64_t sbk, int64_t sbj, double beta, double* __restrict__ C, int64_t ldc) {
    __shared__ double As[DG_BK][DG_BM + DG_PAD];
    __shared__ double Bs[DG_BK][DG_BN + DG_PAD];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = (warp >> 2) * 64, wn = (warp & 3) * 32;  // warp tile origin inside the block tile
    const int i0 = blockIdx.y * DG_BM, j0 = blockIdx.x * DG_BN;
    constexpr int PER = DG_BK * DG_BM / DG_THREADS;  // 8 elements of each operand per thread and k-tile
    double ra[PER], rb[PER];
    auto load_tile = [&](int k0) {
#pragma unroll
        for (int e = 0; e < PER; ++e) {
            const int idx = tid + e * DG_THREADS;
            int kk, ii;
            if (sak == 1) { kk = idx % DG_BK; ii = idx / DG_BK; } else { ii = idx % DG_BM; kk = idx / DG_BM; }
            const int gi = i0 + ii, gk = k0 + kk;
            ra[e] = (gi < M && gk < K) ? A[gi * sai + gk * sak] : 0.0;
            int kb, jj;
            if (sbk == 1) { kb = idx % DG_BK; jj = idx / DG_BK; } else { jj = idx % DG_BN; kb = idx / DG_BN; }
            const int gj = j0 + jj, gkb = k0 + kb;
            rb[e] = (gj < N && gkb < K) ? B[gkb * sbk + gj * sbj] : 0.0;
        }
    };
    auto store_tile = [&] {
#pragma unroll
        for (int e = 0; e < PER; ++e) {
            const int idx = tid + e * DG_THREADS;
            int kk, ii;
            if (sak == 1) { kk = idx % DG_BK; ii = idx / DG_BK; } else { ii = idx % DG_BM; kk = idx / DG_BM; }
            As[kk][ii] = ra[e];
            int kb, jj;
            if (sbk == 1) { kb = idx % DG_BK; jj = idx / DG_BK; } else { jj = idx % DG_BN; kb = idx / DG_BN; }
            Bs[kb][jj] = rb[e];
        }
    };
    double acc[8][4][2] = {};
    const int fr = lane >> 2, fk = lane & 3;  // fragment row / column index, k index
    load_tile(0);
    for (int k0 = 0; k0 < K; k0 += DG_BK) {
        __syncthreads();  // everybody is done with the previous tile
        store_tile();
        __syncthreads();
        if (k0 + DG_BK < K) load_tile(k0 + DG_BK);
#pragma unroll
        for (int ks = 0; ks < DG_BK; ks += 4) {
            double a[8], b[4];
#pragma unroll
            for (int mi = 0; mi < 8; ++mi) a[mi] = As[ks + fk][wm + mi * 8 + fr];
#pragma unroll
            for (int ni = 0; ni < 4; ++ni) b[ni] = Bs[ks + fk][wn + ni * 8 + fr];
#pragma unroll
            for (int mi = 0; mi < 8; ++mi)
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) dmma_m8n8k4(acc[mi][ni][0], acc[mi][ni][1], a[mi], b[ni]);
        }
    }
#pragma unroll
    for (int mi = 0; mi < 8; ++mi) {
        const int gi = i0 + wm + mi * 8 + fr;
        if (gi >= M) continue;
#pragma unroll
        for (int ni = 0; ni < 4; ++ni)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int gj = j0 + wn + ni * 8 + 2 * fk + h;
                if (gj >= N) continue;
                double* p = C + gi * ldc + gj;
                *p = (beta == 0.0) ? alpha * acc[mi][ni][h] : fma(alpha, acc[mi][ni][h], beta * *p);
            }
    }
}

__global__ void k_set_identity(int n, double* __restrict__ A) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < (size_t)n * n) A[i] = (i / n == i % n) ? 1.0 : 0.0;
}

// Unblocked Cholesky of the nb x nb diagonal block at A[k0,k0] (nb <= DENSE_NB), lower triangle; one
// block of DENSE_NB*DENSE_NB threads.  *fail is set if a pivot is not positive.
__global__ void k_potrf_diag(double* __restrict__ A, int64_t lda, int k0, int nb, int* __restrict__ fail) {
    __shared__ double S[DENSE_NB][DENSE_NB + 1];
    const int j = threadIdx.x % DENSE_NB, i = threadIdx.x / DENSE_NB;
    if (i < nb && j < nb) S[i][j] = A[(k0 + i) * lda + k0 + j];
    __syncthreads();
    for (int k = 0; k < nb; ++k) {
        if (i == k && j == k) {
            const double d = S[k][k];
            if (!(d > 0.0)) { *fail = 1; S[k][k] = 1.0; } else S[k][k] = sqrt(d);
        }
        __syncthreads();
        if (j == k && i > k && i < nb) S[i][k] /= S[k][k];
        __syncthreads();
        if (i > k && j > k && j <= i && i < nb) S[i][j] -= S[i][k] * S[j][k];
        __syncthreads();
    }
    if (i < nb && j < nb) A[(k0 + i) * lda + k0 + j] = (j <= i) ? S[i][j] : 0.0;
}

// Panel below the diagonal block: rows i in (k0+nb, n): A[i, k0:k0+nb] <- A[i, k0:k0+nb] L_kk^-T.
__global__ void k_potrf_panel(double* __restrict__ A, int64_t lda, int n, int k0, int nb) {
    __shared__ double S[DENSE_NB][DENSE_NB + 1];
    for (int e = threadIdx.x; e < nb * nb; e += blockDim.x) S[e / nb][e % nb] = A[(k0 + e / nb) * lda + k0 + e % nb];
    __syncthreads();
    const int i = k0 + nb + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double x[DENSE_NB];
    for (int j = 0; j < nb; ++j) {
        double s = A[i * lda + k0 + j];
        for (int l = 0; l < j; ++l) s = fma(-x[l], S[j][l], s);
        x[j] = s / S[j][j];
    }
    for (int j = 0; j < nb; ++j) A[i * lda + k0 + j] = x[j];
}

// Forward panel solve: rows k0..k0+nb of X <- L_kk^-1 B_k ; one thread per right-hand-side column.
__global__ void k_trsm_fwd_diag(const double* __restrict__ L, int64_t lda, int k0, int nb, double* __restrict__ Bm,
                                int64_t ldb, int nrhs) {
    __shared__ double S[DENSE_NB][DENSE_NB + 1];
    for (int e = threadIdx.x; e < nb * nb; e += blockDim.x) S[e / nb][e % nb] = L[(k0 + e / nb) * lda + k0 + e % nb];
    __syncthreads();
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nrhs) return;
    double x[DENSE_NB];
    for (int j = 0; j < nb; ++j) {
        double s = Bm[(k0 + j) * ldb + c];
        for (int l = 0; l < j; ++l) s = fma(-S[j][l], x[l], s);
        x[j] = s / S[j][j];
        Bm[(k0 + j) * ldb + c] = x[j];
    }
}

}  // namespace pdn
