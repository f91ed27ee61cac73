// S1, uniform-tier fast path: the paper's own intra-die kernel.
//
// On a uniform N x N tier (every x-segment g_x, every y-segment g_y) the paper fills the intra-die
// arrays with Wu's closed form, Eq. (3), one thread per entry, an O(N^2) double
// cosine sum each, with partitioned partial sums and a cosine recurrence.  Eq. (3)
// is the spectral expansion of the tier's pseudo-inverse in its DCT-II eigenbasis
//     L^+[u,v] = sum_{(a,b) != 0} phi_a(x_u) phi_b(y_u) phi_a(x_v) phi_b(y_v) / lambda_ab,
//     phi_a(x) = c_a cos(a pi (x + 1/2) / N), c_0^2 = 1/N, c_a^2 = 2/N,
//     lambda_ab = g_x (2 - 2 cos(a pi / N)) + g_y (2 - 2 cos(b pi / N)),
// and R_jk = Z_jj + Z_kk - 2 Z_jk with Z = L^+ gives back Eq. (3).  Instead of repeating the O(N^2)
// sum for each of the ~10^6 entries, the product-to-sum identity cos A cos B = (cos(A-B) + cos(A+B))/2
// turns every entry into FOUR look-ups in one table per tier,
//     L^+[u,v] = 1/4 ( G[|x_u-x_v|][|y_u-y_v|] + G[|x_u-x_v|][y_u+y_v+1]
//                    + G[x_u+x_v+1][|y_u-y_v|] + G[x_u+x_v+1][y_u+y_v+1] ),
//     G[t][s] = sum_{(a,b) != 0} W_ab cos(a pi t / N) cos(b pi s / N),   W_ab = c_a^2 c_b^2 / lambda_ab,
// for t, s in [0, 2N), and the table is two dense FP64 contractions  T = W C^T,  G = C T  with the
// 2N x N cosine matrix C[t][a] = cos(pi (a t mod 2N) / N) (exact argument reduction in integers): the
// paper's "partial sums computed in parallel, summed after" becomes GEMM tiling.  12 N^3 flops per
// tier (13 GFLOP at N = 1024) replace all port solves of that tier.
#pragma once
#include "common.cuh"

namespace pdn {

// flag[0] = 1 if some present x-segment differs from gx[0] or some y-segment from gy[0] (or is absent).
__global__ void k_uniform_check(int n, int pitch, const double* __restrict__ gx, const double* __restrict__ gy,
                                int* __restrict__ flag) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = false;
    if (i < n * pitch) {
        const int y = i / pitch, x = i % pitch;
        if (x < n) {
            const double g0x = gx[0], g0y = gy[0];
            if (x < n - 1 && gx[i] != g0x) bad = true;
            if (y < n - 1 && gy[i] != g0y) bad = true;
        }
    }
    // every writer stores the same value: a plain store by one lane per warp (on a non-uniform tier nearly every
    // thread finds a difference, and a million atomics on one word took 0.7 ms)
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) *flag = 1;
}

// C[t][a] = cos(pi (a t mod 2N) / N),  t in [0, 2N), a in [0, N)
__global__ void k_cos_matrix(int n, double* __restrict__ C) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)2 * n * n) return;
    const int t = (int)(i / n), a = (int)(i % n);
    const long long m = ((long long)a * t) % (2LL * n);
    C[i] = cospi((double)m / (double)n);
}

// W[a][b] = c_a^2 c_b^2 / lambda_ab  (0 for the constant mode a = b = 0)
__global__ void k_spectral_weights(int n, double g_x, double g_y, double* __restrict__ W) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)n * n) return;
    const int a = (int)(i / n), b = (int)(i % n);
    if (a == 0 && b == 0) { W[i] = 0.0; return; }
    // 2 - 2 cos(theta) = 4 sin^2(theta / 2): no cancellation for the low modes
    const double sa = sinpi(0.5 * (double)a / (double)n), sb = sinpi(0.5 * (double)b / (double)n);
    const double lam = 4.0 * (g_x * sa * sa + g_y * sb * sb);
    const double ca = (a == 0 ? 1.0 : 2.0) / (double)n, cb = (b == 0 ? 1.0 : 2.0) / (double)n;
    W[i] = ca * cb / lam;
}

__device__ __forceinline__ double uniform_pinv_entry(const double* __restrict__ G, int n, int pitch, int u, int v) {
    const int yu = u / pitch, xu = u % pitch, yv = v / pitch, xv = v % pitch;
    const int dx = abs(xu - xv), dy = abs(yu - yv), sx = xu + xv + 1, sy = yu + yv + 1;
    const size_t ld = (size_t)2 * n;
    return 0.25 * ((G[dx * ld + dy] + G[sx * ld + sy]) + (G[dx * ld + sy] + G[sx * ld + dy]));
}

// ZT[j][k] = L^+[port j, port k] for the rows j < nrows (the TSV ports; all ports with PDN_TERMINAL_PAIRS)
// against all ports k < q (grid.y walks rows 0 .. nrows); zdiag[s] = L^+[s, s] for the terminal ports.  node[] holds
// pitched offsets y*pitch + x; G is indexed [x][y].
__global__ void k_uniform_gather(const double* __restrict__ G, int n, int pitch, const int* __restrict__ node, int ntsv,
                                 int nrows, int q, double* __restrict__ ZT, double* __restrict__ zdiag) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= q) return;
    for (int j = blockIdx.y; j <= nrows; j += gridDim.y) {
        if (j < nrows) ZT[(size_t)j * q + k] = uniform_pinv_entry(G, n, pitch, node[j], node[k]);
        else if (k >= ntsv) zdiag[k - ntsv] = uniform_pinv_entry(G, n, pitch, node[k], node[k]);
    }
}

}  // namespace pdn
