// S1: batched matrix-free multigrid-PCG kernels on the per-tier 2D 5-point stencil.
//
// All vectors are batched planes  v[b][y][x]  (b = right-hand side, contiguous ny*nx doubles each).
// Every kernel works on overlapped tiles: a block stages the TI x TI tile plus a halo of H nodes in
// shared memory, runs all the sweeps of its multigrid stage there (halo recomputed redundantly, no
// inter-block exchange), and writes only the tile interior.  Nodes outside the mesh hold zeros and
// have zero conductances, so no boundary special-casing is needed inside the sweeps.
#pragma once
#include "common.cuh"

namespace pdn {

constexpr int STENCIL_THREADS = 256;

struct TileGeom {
    int y0, x0;  // global coordinates of extended-tile element (0,0)
    int E;       // extended size
};

// L z at extended-tile element (ey, ex) whose global node (gy, gx) lies inside the mesh.
template <int E>
__device__ __forceinline__ double stencil_apply(const Level& L, const double* __restrict__ sz, int ey, int ex,
                                                int gy, int gx) {
    const int gi = gy * L.nx + gx;
    const double zc = sz[ey * E + ex];
    const double gE = __ldg(L.gx + gi);
    const double gS = __ldg(L.gy + gi);
    const double gW = gx > 0 ? __ldg(L.gx + gi - 1) : 0.0;
    const double gN = gy > 0 ? __ldg(L.gy + gi - L.nx) : 0.0;
    double a = gE * (zc - sz[ey * E + ex + 1]);
    a = fma(gW, zc - sz[ey * E + ex - 1], a);
    a = fma(gS, zc - sz[(ey + 1) * E + ex], a);
    a = fma(gN, zc - sz[(ey - 1) * E + ex], a);
    return a;
}

// One Chebyshev step k on the region [lo, E-lo)^2:  d = c1 d + c2 dinv (r - L z);  then z += d.
template <int E>
__device__ __forceinline__ void cheb_step(const Level& L, const double* sr, double* sz, double* sd, int y0, int x0,
                                          int lo, double c1, double c2) {
    const int W = E - 2 * lo;
    for (int i = threadIdx.x; i < W * W; i += STENCIL_THREADS) {
        const int ey = lo + i / W, ex = lo + i % W;
        const int gy = y0 + ey, gx = x0 + ex;
        double d = 0.0;
        if (gy >= 0 && gy < L.ny && gx >= 0 && gx < L.nx) {
            const double res = sr[ey * E + ex] - stencil_apply<E>(L, sz, ey, ex, gy, gx);
            d = fma(c1, sd[ey * E + ex], c2 * __ldg(L.dinv + gy * L.nx + gx) * res);
        }
        sd[ey * E + ex] = d;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < W * W; i += STENCIL_THREADS) {
        const int ey = lo + i / W, ex = lo + i % W;
        sz[ey * E + ex] += sd[ey * E + ex];
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------
// Down stage of the V-cycle on level L (optionally fused with the CG residual update on level 0):
//   [r = r_in - alpha q ; rr += r.r]   z = Cheb_nu(0, r)   rc = R (r - L z)
// R = sum over the 2x2 aggregate (transpose of piecewise-constant prolongation).
// grid = (tiles_x, tiles_y, B); dynamic smem = 3 * E * E doubles, E = TI + 2 nu.
template <int TI, int NU>
__global__ void __launch_bounds__(STENCIL_THREADS)
k_down(Level L, Cheb ch, const double* __restrict__ r_in, const double* __restrict__ q,
       const double* __restrict__ alpha, double* __restrict__ r_out, double* __restrict__ z_out,
       double* __restrict__ rc, int cny, int cnx, double* __restrict__ rr_acc) {
    constexpr int H = NU, E = TI + 2 * H;
    extern __shared__ double smem[];
    double* sr = smem;
    double* sz = smem + E * E;
    double* sd = smem + 2 * E * E;
    __shared__ double red[32];
    const int b = blockIdx.z;
    const size_t plane = (size_t)L.ny * L.nx;
    const int y0 = blockIdx.y * TI - H, x0 = blockIdx.x * TI - H;
    const double* rb = r_in + b * plane;
    const double a = q ? alpha[b] : 0.0;
    double rr = 0.0;
    for (int i = threadIdx.x; i < E * E; i += STENCIL_THREADS) {
        const int ey = i / E, ex = i % E;
        const int gy = y0 + ey, gx = x0 + ex;
        double v = 0.0, dv = 0.0;
        if (gy >= 0 && gy < L.ny && gx >= 0 && gx < L.nx) {
            const size_t gi = (size_t)gy * L.nx + gx;
            v = rb[gi];
            if (q) {
                v = fma(-a, q[b * plane + gi], v);
                if (ey >= H && ey < H + TI && ex >= H && ex < H + TI) {
                    r_out[b * plane + gi] = v;
                    rr = fma(v, v, rr);
                }
            }
            dv = ch.c2[0] * __ldg(L.dinv + gi) * v;
        }
        sr[i] = v;
        sd[i] = dv;
        sz[i] = dv;
    }
    __syncthreads();
#pragma unroll
    for (int k = 1; k < NU; ++k) cheb_step<E>(L, sr, sz, sd, y0, x0, k, ch.c1[k], ch.c2[k]);
    // write z (interior)
    for (int i = threadIdx.x; i < TI * TI; i += STENCIL_THREADS) {
        const int ey = H + i / TI, ex = H + i % TI;
        const int gy = y0 + ey, gx = x0 + ex;
        if (gy < L.ny && gx < L.nx) z_out[b * plane + (size_t)gy * L.nx + gx] = sz[ey * E + ex];
    }
    // residual + restriction: one thread per coarse cell of the tile
    constexpr int TC = TI / 2;
    for (int i = threadIdx.x; i < TC * TC; i += STENCIL_THREADS) {
        const int cy = i / TC, cx = i % TC;
        const int gcy = blockIdx.y * TC + cy, gcx = blockIdx.x * TC + cx;
        if (gcy >= cny || gcx >= cnx) continue;
        double s = 0.0;
#pragma unroll
        for (int dy = 0; dy < 2; ++dy)
#pragma unroll
            for (int dx = 0; dx < 2; ++dx) {
                const int ey = H + 2 * cy + dy, ex = H + 2 * cx + dx;
                const int gy = y0 + ey, gx = x0 + ex;
                if (gy < L.ny && gx < L.nx) s += sr[ey * E + ex] - stencil_apply<E>(L, sz, ey, ex, gy, gx);
            }
        rc[(size_t)b * cny * cnx + (size_t)gcy * cnx + gcx] = s;
    }
    if (q) {
        rr = block_sum(rr, red);
        if (threadIdx.x == 0) atomicAdd(rr_acc + b, rr);
    }
}

// ---------------------------------------------------------------------------------------------
// Up stage on level L:  z = z_in + P e_c ;  z = Cheb_nu(z, r) ;  [rz += r.z on level 0]
// P = piecewise-constant prolongation (fine (y,x) takes coarse (y/2, x/2)).
template <int TI, int NU>
__global__ void __launch_bounds__(STENCIL_THREADS)
k_up(Level L, Cheb ch, const double* __restrict__ r, const double* __restrict__ z_in,
     const double* __restrict__ ec, int cny, int cnx, double* __restrict__ z_out, double* __restrict__ rz_acc) {
    constexpr int H = NU, E = TI + 2 * H;
    extern __shared__ double smem[];
    double* sr = smem;
    double* sz = smem + E * E;
    double* sd = smem + 2 * E * E;
    __shared__ double red[32];
    const int b = blockIdx.z;
    const size_t plane = (size_t)L.ny * L.nx;
    const size_t cplane = (size_t)cny * cnx;
    const int y0 = blockIdx.y * TI - H, x0 = blockIdx.x * TI - H;
    for (int i = threadIdx.x; i < E * E; i += STENCIL_THREADS) {
        const int ey = i / E, ex = i % E;
        const int gy = y0 + ey, gx = x0 + ex;
        double rv = 0.0, zv = 0.0;
        if (gy >= 0 && gy < L.ny && gx >= 0 && gx < L.nx) {
            const size_t gi = (size_t)gy * L.nx + gx;
            rv = r[b * plane + gi];
            zv = z_in[b * plane + gi] + ec[b * cplane + (size_t)(gy >> 1) * cnx + (gx >> 1)];
        }
        sr[i] = rv;
        sz[i] = zv;
        sd[i] = 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NU; ++k) cheb_step<E>(L, sr, sz, sd, y0, x0, k + 1, ch.c1[k], ch.c2[k]);
    double rz = 0.0;
    for (int i = threadIdx.x; i < TI * TI; i += STENCIL_THREADS) {
        const int ey = H + i / TI, ex = H + i % TI;
        const int gy = y0 + ey, gx = x0 + ex;
        if (gy < L.ny && gx < L.nx) {
            const double zv = sz[ey * E + ex];
            z_out[b * plane + (size_t)gy * L.nx + gx] = zv;
            rz = fma(sr[ey * E + ex], zv, rz);
        }
    }
    if (rz_acc) {
        rz = block_sum(rz, red);
        if (threadIdx.x == 0) atomicAdd(rz_acc + b, rz);
    }
}

// ---------------------------------------------------------------------------------------------
// CG direction update fused with the operator apply (level 0):
//   p = z + beta p_old ;  q = L p ;  pq += p.q ;  sump += sum(p)
template <int TI>
__global__ void __launch_bounds__(STENCIL_THREADS)
k_pq(Level L, const double* __restrict__ z, const double* __restrict__ p_old, const double* __restrict__ beta,
     double* __restrict__ p_new, double* __restrict__ q, double* __restrict__ pq_acc, double* __restrict__ sump_acc) {
    constexpr int H = 1, E = TI + 2 * H;
    __shared__ double sp[E * E];
    __shared__ double red[32];
    const int b = blockIdx.z;
    const size_t plane = (size_t)L.ny * L.nx;
    const int y0 = blockIdx.y * TI - H, x0 = blockIdx.x * TI - H;
    const double bt = beta[b];
    for (int i = threadIdx.x; i < E * E; i += STENCIL_THREADS) {
        const int ey = i / E, ex = i % E;
        const int gy = y0 + ey, gx = x0 + ex;
        double v = 0.0;
        if (gy >= 0 && gy < L.ny && gx >= 0 && gx < L.nx) {
            const size_t gi = b * plane + (size_t)gy * L.nx + gx;
            v = z[gi];
            if (bt != 0.0) v = fma(bt, p_old[gi], v);
        }
        sp[i] = v;
    }
    __syncthreads();
    double pq = 0.0, sp_sum = 0.0;
    for (int i = threadIdx.x; i < TI * TI; i += STENCIL_THREADS) {
        const int ey = H + i / TI, ex = H + i % TI;
        const int gy = y0 + ey, gx = x0 + ex;
        if (gy < L.ny && gx < L.nx) {
            const double pv = sp[ey * E + ex];
            const double qv = stencil_apply<E>(L, sp, ey, ex, gy, gx);
            const size_t gi = b * plane + (size_t)gy * L.nx + gx;
            p_new[gi] = pv;
            q[gi] = qv;
            pq = fma(pv, qv, pq);
            sp_sum += pv;
        }
    }
    pq = block_sum(pq, red);
    if (threadIdx.x == 0) atomicAdd(pq_acc + b, pq);
    sp_sum = block_sum(sp_sum, red);
    if (threadIdx.x == 0) atomicAdd(sump_acc + b, sp_sum);
}

// Coarsest level: e = pinv * r, one thread per (b, i); nc = ny*nx <= 16.
__global__ void k_coarse_pinv(const double* __restrict__ pinv, int nc, const double* __restrict__ r,
                              double* __restrict__ e, int B) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= B * nc) return;
    const int b = t / nc, i = t % nc;
    double s = 0.0;
    for (int j = 0; j < nc; ++j) s = fma(__ldg(pinv + i * nc + j), r[(size_t)b * nc + j], s);
    e[t] = s;
}

}  // namespace pdn
