// Shared device-side definitions of the PDN effective-resistance path (sm_100a only).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace pdn {

constexpr int MAX_NU = 8;       // max smoothing steps per side
constexpr int MAX_LEVELS = 16;  // multigrid levels (n halves per level)
constexpr int COARSEST_MAX = 4; // coarsest level has n <= 4 (<= 16 unknowns, dense pseudo-inverse)

// One multigrid level of one tier: matrix-free 5-point stencil with per-edge conductances.
//
// Every plane and every batched vector of a level is stored with a row pitch of `pitch` doubles
// (nx rounded up to an even number), so that a thread's two adjacent columns are one aligned
// 16-byte word and TMA row strides are multiples of 16 bytes.  Pad entries of planes are zero.
//
// The V-cycle works on the symmetrically scaled operator  A^ = S L S ~ I - N  (S = D^-1/2), so that the
// Jacobi-preconditioned Richardson step z <- z + w D^-1 (r - L z) becomes, for y = z/s, r^ = s r:
//   y <- (1-w) y + w (r^ + sum_nb h_nb y_nb)      -- no diagonal in the inner loop.
//   sc[y][x]  = (s, sd) = (1/sqrt(d), sqrt(d)) rounded to FP32 (d = sum of the incident conductances;
//               (0, 0) for a node with d = 0).  The scaling is part of the PRECONDITIONER only: any
//               positive diagonal works there, symmetry needs the same S on the way in (r^ = s r,
//               rc = R sd res) and out (y += sd P e, z = s y), and FP32 entries halve the on-chip
//               footprint.  All arithmetic with them is FP64.
//   hE[y][x]  = gx[y][x] * s[y][x] * s[y][x+1],  hS[y][x] = gy[y][x] * s[y][x] * s[y+1][x]   (FP64).
// The CG operator apply (k_pq3) uses the raw gx / gy.
struct Level {
    int ny, nx, pitch;
    const double* gx;   // raw conductances (level 0: sanitised copy of the caller's planes)
    const double* gy;
    const double* hE;
    const double* hS;
    const float2* sc;
};

// Richardson steps with the reciprocals of the Chebyshev nodes of [2/ratio, 2] as step lengths: the
// same polynomial as nu Chebyshev semi-iteration steps on D^-1 L (lambda_max(D^-1 L) <= 2 for any
// graph Laplacian), with no direction vector to carry.
struct ChebR {
    int nu;
    double w[MAX_NU];
};

// Per-right-hand-side PCG scalars of one batch (device arrays of length B).
struct PcgScalars {
    double* rho;     // r.z of the current iteration
    double* rz;      // accumulator: r.z after the V-cycle
    double* pq;      // accumulator: z.Lz of this iteration (k_pq3)
    double* rr;      // accumulator: ||r||^2
    double* sump;    // accumulator: sum(z) of this iteration (k_pq3)
    double* pap;     // p.Lp of the current direction, by recurrence: z.Lz - beta^2 p_old.Lp_old
    double* psum;    // sum(p) of the current direction, by recurrence: sum(z) + beta sum(p_old)
    double* alpha;
    double* beta;
    double* qq;      // accumulator: ||q||^2 of this iteration (k_pq3_last only)
    double* rq;      // accumulator: r.q of this iteration (k_pq3_last only)
    double* rrk;     // ||r_k||^2 as of the last convergence check
    double* arho;    // sum_j alpha_j rho_j = ||x_k - x_0||_L^2 (Hestenes-Stiefel): the energy a terminal solve has gained
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

// ---------------------------------------------------------------------------------------------
// TMA (cp.async.bulk.tensor) + mbarrier wrappers.  Tiles with halos are fetched as 3D boxes
// (x, y, right-hand side) of a tensor map; coordinates may be negative or run past the mesh:
// out-of-bounds elements arrive as zeros, which is exactly the "no node, no conductance" padding
// the sweeps need.
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2,
                                            uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(smem_dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(smem_u32(smem_dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}

}  // namespace pdn
