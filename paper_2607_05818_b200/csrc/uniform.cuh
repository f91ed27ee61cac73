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
// turns every entry into FOUR look-ups in one table,
//     L^+[u,v] = 1/4 ( G[|y_u-y_v|][|x_u-x_v|] + G[f(y_u+y_v+1)][f(x_u+x_v+1)]
//                    + G[|y_u-y_v|][f(x_u+x_v+1)] + G[f(y_u+y_v+1)][|x_u-x_v|] ),
//     G[t][s] = sum_{(a,b) != 0} W_ab cos(a pi t / N) cos(b pi s / N),   W_ab = c_a^2 c_b^2 / lambda_ab
// (a = mode along y, b = mode along x; the table is indexed [y][x] so that nodes of one mesh row read consecutive
// entries), for t, s in [0, N]: cos(a pi t / N) is even about t = N, so an argument t in (N, 2N) folds to
// f(t) = 2N - t.  The table is two dense FP64 contractions  T = W C^T,  G = C T  with the (N+1) x N cosine matrix
// C[t][a] = cos(pi a t / N) (exact argument reduction in integers): the paper's "partial sums computed in parallel,
// summed after" becomes GEMM tiling.  4 N^3 flops per table (4.3 GFLOP at N = 1024).  The table depends on the
// segment conductances only through rho = g_x / g_y and a scale: G(g_x, g_y) = G(rho, 1) / g_y, so tiers that differ
// by a factor (BASELINE's r_t = c (t+1)) share one table.
//
// Two uses: (i) a uniform tier is reduced whole from the table (all its port solves replaced by a gather);
// (ii) on a NON-uniform tier whose segments scatter around a mean (BASELINE's +-10 % jitter, removed segments), the
// same closed form with the mean conductances is the INITIAL GUESS x0 of every port solve ("can be
// easily computed using Eq. (3)"): PCG then starts from r0 = b - L x0 = (L_mean - L) x0, about a decade below
// ||b||, and the gathered result is x0[port] + the PCG correction (guess.cuh).
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

// C[t][a] = cos(pi (a t mod 2N) / N),  t in [0, N], a in [0, N)
__global__ void k_cos_matrix(int n, double* __restrict__ C) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)(n + 1) * n) return;
    const int t = (int)(i / n), a = (int)(i % n);
    const long long m = ((long long)a * t) % (2LL * n);
    C[i] = cospi((double)m / (double)n);
}

// W[a][b] = c_a^2 c_b^2 / lambda_ab  (0 for the constant mode a = b = 0); a = mode along y, b = mode along x
__global__ void k_spectral_weights(int n, double g_x, double g_y, double* __restrict__ W) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)n * n) return;
    const int a = (int)(i / n), b = (int)(i % n);
    if (a == 0 && b == 0) { W[i] = 0.0; return; }
    // 2 - 2 cos(theta) = 4 sin^2(theta / 2): no cancellation for the low modes
    const double sa = sinpi(0.5 * (double)a / (double)n), sb = sinpi(0.5 * (double)b / (double)n);
    const double lam = 4.0 * (g_y * sa * sa + g_x * sb * sb);
    const double ca = (a == 0 ? 1.0 : 2.0) / (double)n, cb = (b == 0 ? 1.0 : 2.0) / (double)n;
    W[i] = ca * cb / lam;
}

// (L_mean^+)[node (yu, xu), node (yv, xv)] from the table (leading dimension n + 1); TG = double or float
template <class TG>
__device__ __forceinline__ double spectral_entry(const TG* __restrict__ G, int n, int yu, int xu, int yv, int xv) {
    const int dx = abs(xu - xv), dy = abs(yu - yv);
    int sx = xu + xv + 1, sy = yu + yv + 1;
    sx = sx <= n ? sx : 2 * n - sx;
    sy = sy <= n ? sy : 2 * n - sy;
    const size_t ld = (size_t)n + 1;
    return 0.25 * (((double)G[dy * ld + dx] + (double)G[sy * ld + sx]) + ((double)G[dy * ld + sx] + (double)G[sy * ld + dx]));
}

__device__ __forceinline__ double uniform_pinv_entry(const double* __restrict__ G, double scale, int n, int pitch, int u, int v) {
    return scale * spectral_entry<double>(G, n, u / pitch, u % pitch, v / pitch, v % pitch);
}

// ZT[j][k] = L^+[port j, port k] for the rows j < nrows (the TSV ports; all ports with PDN_TERMINAL_PAIRS)
// against all ports k < q (grid.y walks rows 0 .. nrows); zdiag[s] = L^+[s, s] for the terminal ports.  node[] holds
// pitched offsets y*pitch + x; G is the table of (rho, 1), scale = 1 / g_y.
__global__ void k_uniform_gather(const double* __restrict__ G, double scale, int n, int pitch, const int* __restrict__ node, int ntsv,
                                 int nrows, int q, double* __restrict__ ZT, double* __restrict__ zdiag) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= q) return;
    for (int j = blockIdx.y; j <= nrows; j += gridDim.y) {
        if (j < nrows) ZT[(size_t)j * q + k] = uniform_pinv_entry(G, scale, n, pitch, node[j], node[k]);
        else if (k >= ntsv) zdiag[k - ntsv] = uniform_pinv_entry(G, scale, n, pitch, node[k], node[k]);
    }
}

// FP32 copy of a table: the initial guess needs no more (the PCG correction absorbs whatever the guess lacks, as
// long as the SAME x0 enters r0 = b - L x0 and the gathered result), and it halves the L2 traffic of guess.cuh.
__global__ void k_table_to_float(size_t cnt, const double* __restrict__ G, float* __restrict__ Gf) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < cnt) Gf[i] = (float)G[i];
}

// The same FP32 values with a row pitch of `pitch` floats (a multiple of four: TMA row strides are multiples of 16
// bytes), pads zero: the table the window fetches of k_guess_rhs read.
__global__ void k_table_to_pitched(int n, int pitch, const double* __restrict__ G, float* __restrict__ Gq) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)(n + 1) * pitch) return;
    const size_t t = i / pitch, s = i % pitch;
    Gq[i] = s <= (size_t)n ? (float)G[t * (n + 1) + s] : 0.f;
}

}  // namespace pdn
