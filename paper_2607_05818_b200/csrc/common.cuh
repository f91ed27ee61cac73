// Shared device-side definitions of the PDN effective-resistance path (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pdn {

constexpr int MAX_NU = 8;       // max Chebyshev steps per side
constexpr int MAX_LEVELS = 16;  // multigrid levels (n halves per level)
constexpr int COARSEST_MAX = 4; // coarsest level has n <= 4 (<= 16 unknowns, dense pseudo-inverse)

// One multigrid level of one tier: matrix-free 5-point stencil with per-edge conductances.
//   gx[y*nx+x] joins (y,x)-(y,x+1), zero in the last column; gy[y*nx+x] joins (y,x)-(y+1,x), zero in
//   the last row; dinv = 1 / (sum of the incident conductances) (0 for an isolated node).
struct Level {
    int ny, nx;
    const double* gx;
    const double* gy;
    const double* dinv;
};

// Chebyshev polynomial smoother on D^-1 L with spectrum bound [2/ratio, 2] (lambda_max(D^-1 L) <= 2
// for any graph Laplacian):  d_0 = c2[0] D^-1 res_0;  d_k = c1[k] d_{k-1} + c2[k] D^-1 res_k;  z += d_k.
struct Cheb {
    int nu;
    double c1[MAX_NU];
    double c2[MAX_NU];
};

// Per-right-hand-side PCG scalars of one batch (device arrays of length B).
struct PcgScalars {
    double* rho;     // r.z of the current iteration
    double* rz;      // accumulator: r.z after the V-cycle
    double* pq;      // accumulator: p.Lp
    double* rr;      // accumulator: ||r||^2
    double* sump;    // accumulator: sum(p)
    double* alpha;
    double* beta;
    double* xmean;   // mean of the (implicit) solution x = sum_k alpha_k p_k
    double* relres;  // ||r|| / ||b|| at the last check
    int* active;     // 1 while the right-hand side has not converged
    int* n_active;   // single int: number of active right-hand sides
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Block-wide sum; result valid in thread 0.  `scratch` holds >= 32 doubles.
__device__ __forceinline__ double block_sum(double v, double* scratch) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) scratch[w] = v;
    __syncthreads();
    if (w == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        v = lane < nw ? scratch[lane] : 0.0;
        v = warp_sum(v);
    }
    return v;
}

}  // namespace pdn
