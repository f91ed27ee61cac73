// S0: tier representation -- sanitised copies of the conductance planes, the multigrid hierarchy
// (2x2 aggregation, coarse conductance = 1/2 * sum of the two fine segments crossing the coarse
// face), the symmetric scaling of every level, and the dense pseudo-inverse of the coarsest level.
#pragma once
#include "common.cuh"

namespace pdn {

// Copy the caller's dense n x n planes into pitched planes, zero the padding column / row, flag bad
// values (negative, NaN, inf).
__global__ void k_import_planes(const double* __restrict__ gx_in, const double* __restrict__ gy_in, int n, int pitch,
                                double* __restrict__ gx, double* __restrict__ gy, int* __restrict__ bad) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * pitch) return;
    const int y = i / pitch, x = i % pitch;
    double a = 0.0, b = 0.0;
    if (x < n) {
        a = x < n - 1 ? gx_in[y * n + x] : 0.0;
        b = y < n - 1 ? gy_in[y * n + x] : 0.0;
        if (!(a >= 0.0) || !(b >= 0.0) || isinf(a) || isinf(b)) {
            atomicExch(bad, 1);
            a = 0.0;
            b = 0.0;
        }
    }
    gx[i] = a;
    gy[i] = b;
}

// sums[0] += sum of the x-conductances, sums[1] += sum of the y-conductances (the tier's anisotropy, which
// picks the smoothing interval of the Chebyshev polynomial; pdn_api.cu), sums[2], sums[3] += the sums of their
// squares (how far the tier is from its mean mesh: whether the closed-form initial guess is worth trying).
__global__ void k_plane_sums(int n_elems, const double* __restrict__ gx, const double* __restrict__ gy,
                             double* __restrict__ sums) {
    __shared__ double red[32];
    double a = 0.0, b = 0.0, a2 = 0.0, b2 = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_elems; i += gridDim.x * blockDim.x) {
        const double u = gx[i], v = gy[i];
        a += u; b += v;
        a2 = fma(u, u, a2); b2 = fma(v, v, b2);
    }
    a = block_sum(a, red);
    if (threadIdx.x == 0) atomicAdd(sums, a);
    b = block_sum(b, red);
    if (threadIdx.x == 0) atomicAdd(sums + 1, b);
    a2 = block_sum(a2, red);
    if (threadIdx.x == 0) atomicAdd(sums + 2, a2);
    b2 = block_sum(b2, red);
    if (threadIdx.x == 0) atomicAdd(sums + 3, b2);
}

// sc = (s, sd) = (1/sqrt(d), sqrt(d)) in FP32, d = sum of incident conductances ((0,0) if the node is
// isolated; flagged on the finest level).
__global__ void k_scale_nodes(int ny, int nx, int pitch, const double* __restrict__ gx, const double* __restrict__ gy,
                              float2* __restrict__ sc, int* __restrict__ isolated) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ny * pitch) return;
    const int y = i / pitch, x = i % pitch;
    double d = 0.0;
    if (x < nx) {
        d = gx[i] + gy[i];
        if (x > 0) d += gx[i - 1];
        if (y > 0) d += gy[i - pitch];
    }
    if (d > 0.0) {
        const double r = sqrt(d);
        sc[i] = make_float2((float)(1.0 / r), (float)r);
    } else {
        sc[i] = make_float2(0.f, 0.f);
        if (isolated && x < nx) atomicExch(isolated, 1);
    }
}

// hE = gx s s_east, hS = gy s s_south  (symmetric scaling with the FP32-rounded s, products in FP64;
// zero where the segment is absent).
__global__ void k_scale_edges(int ny, int nx, int pitch, const double* __restrict__ gx, const double* __restrict__ gy,
                              const float2* __restrict__ sc, double* __restrict__ hE, double* __restrict__ hS) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ny * pitch) return;
    const int y = i / pitch, x = i % pitch;
    const double s = (double)sc[i].x;
    hE[i] = (x + 1 < nx) ? gx[i] * s * (double)sc[i + 1].x : 0.0;
    hS[i] = (x < nx && y + 1 < ny) ? gy[i] * s * (double)sc[i + pitch].x : 0.0;
}

// Coarse planes (cny x cnx, cn = ceil(n/2)) from fine planes (ny x nx).
//   cgx[Y][X] = 1/2 (gx[2Y][2X+1] + gx[2Y+1][2X+1])   -- the fine x-segments leaving aggregate X to X+1
//   cgy[Y][X] = 1/2 (gy[2Y+1][2X] + gy[2Y+1][2X+1])
__global__ void k_coarsen(int ny, int nx, int pitch, const double* __restrict__ gx, const double* __restrict__ gy,
                          int cny, int cnx, int cpitch, double* __restrict__ cgx, double* __restrict__ cgy) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cny * cpitch) return;
    const int Y = i / cpitch, X = i % cpitch;
    double a = 0.0, b = 0.0;
    const int fx = 2 * X + 1, fy = 2 * Y + 1;
    if (X < cnx) {
        if (fx < nx - 1) {  // a segment from column fx to fx+1 exists only if fx+1 < nx
            a += gx[(2 * Y) * pitch + fx];
            if (fy < ny) a += gx[fy * pitch + fx];
        }
        if (fy < ny - 1) {
            b += gy[fy * pitch + 2 * X];
            if (fx < nx) b += gy[fy * pitch + fx];
        }
    }
    cgx[i] = 0.5 * a;
    cgy[i] = 0.5 * b;
}

// Dense pseudo-inverse of the coarsest Laplacian (nc = ny*nx <= 16 unknowns), one warp, lane j owns
// column j of the augmented matrix [L + 11^T/nc | I]:
//   L^+ = (L + 11^T/nc)^-1 - 11^T/nc   (Gauss-Jordan on an SPD matrix, no pivoting needed).
__global__ void k_coarsest_pinv(int ny, int nx, int pitch, const double* __restrict__ gx,
                                const double* __restrict__ gy, double* __restrict__ pinv) {
    __shared__ double A[16][33];
    const int nc = ny * nx, j = threadIdx.x;  // blockDim.x == 32 >= 2 nc
    for (int i = 0; i < nc; ++i) A[i][j] = (j < nc ? 1.0 / nc : (j - nc == i ? 1.0 : 0.0));
    __syncwarp();
    if (j == 0) {
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const int i = y * nx + x;
                if (x < nx - 1) {
                    const double g = gx[y * pitch + x];
                    A[i][i] += g; A[i + 1][i + 1] += g; A[i][i + 1] -= g; A[i + 1][i] -= g;
                }
                if (y < ny - 1) {
                    const double g = gy[y * pitch + x];
                    A[i][i] += g; A[i + nx][i + nx] += g; A[i][i + nx] -= g; A[i + nx][i] -= g;
                }
            }
    }
    __syncwarp();
    for (int k = 0; k < nc; ++k) {
        const double inv = 1.0 / A[k][k];
        __syncwarp();
        const double akj = A[k][j] * inv;
        A[k][j] = akj;
        __syncwarp();
        for (int i = 0; i < nc; ++i) {
            if (i == k) continue;
            const double f = A[i][k];
            __syncwarp();
            A[i][j] -= f * akj;
            __syncwarp();
        }
    }
    if (j < nc)
        for (int i = 0; i < nc; ++i) pinv[i * nc + j] = A[i][nc + j] - 1.0 / nc;
}

// Connectivity of one tier by label propagation: lab[i] = min over the component of the node ids.
// One sweep relaxes every node against its 4 neighbours through existing segments and then follows
// label pointers (pointer jumping); `changed` is set if any label moved.
__global__ void k_label_init(int n2, int* __restrict__ lab) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n2) lab[i] = i;
}

__global__ void k_label_sweep(int ny, int nx, int pitch, const double* __restrict__ gx,
                              const double* __restrict__ gy, int* __restrict__ lab, int* __restrict__ changed) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ny * nx) return;
    const int y = i / nx, x = i % nx;
    const int g = y * pitch + x;
    int m = lab[i];
    const int m0 = m;
    if (x < nx - 1 && gx[g] > 0.0) m = min(m, lab[i + 1]);
    if (x > 0 && gx[g - 1] > 0.0) m = min(m, lab[i - 1]);
    if (y < ny - 1 && gy[g] > 0.0) m = min(m, lab[i + nx]);
    if (y > 0 && gy[g - pitch] > 0.0) m = min(m, lab[i - nx]);
    // pointer jumping: the label of my label is at least as small
    int mm = lab[m];
    while (mm < m) { m = mm; mm = lab[m]; }
    if (m < m0) {
        atomicMin(lab + i, m);
        atomicMin(lab + m0, m);  // pull my old root down too (union by min)
        *changed = 1;
    }
}

__global__ void k_label_check(int n2, const int* __restrict__ lab, int* __restrict__ nonzero) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n2 && lab[i] != 0) *nonzero = 1;
}

}  // namespace pdn
