// S1b, coarse tail of the V-cycle: every multigrid level of at most TAIL_MAX_N x TAIL_MAX_N nodes, down to the
// 4 x 4 pseudo-inverse and back up, in ONE kernel and entirely in shared memory.
//
// On those levels a 64 x 72 register tile (stencil3.cuh) is mostly halo and a launch per level and direction is
// mostly launch latency: at 1024^2 the levels 32^2 .. 4^2 cost 8 launches per cycle, at 128^2 they are most of
// the iteration, and a 32^2 tier is nothing else.  Here a block of TAIL_THREADS threads keeps the coefficients
// of all tail levels resident (loaded once, reused for the G right-hand sides it loops over) and the vectors of
// one right-hand side in zero-bordered arrays, so the sweeps need no boundary cases; same arithmetic as
// k_down3 / k_up3: scaled Richardson steps y <- (1-w) y + w (r^ + N y), residual restricted over 2x2
// aggregates with the sd weights, piecewise-constant prolongation, z = s y.
#pragma once
#include "common.cuh"

namespace pdn {

constexpr int TAIL_MAX_N = 32, TAIL_MAX_LEVELS = 4, TAIL_THREADS = 256;

struct TailParams {
    int nlev;                     // levels in the tail, finest first; the last one is the dense coarsest level
    Level lev[TAIL_MAX_LEVELS];
    const double* pinv;           // (ny*nx)^2 pseudo-inverse of the last level
    ChebR ch;
};

// doubles of shared memory the kernel needs (host and device agree through this function)
__host__ __device__ inline size_t tail_smem_doubles(const TailParams& P) {
    size_t n = 0;
    for (int l = 0; l + 1 < P.nlev; ++l) n += (size_t)7 * (P.lev[l].ny + 2) * (P.lev[l].nx + 2);
    return n + 16 + 16 + 256;
}

// z_out[b] = M_tail^-1 r_in[b] on level P.lev[0] (pitched planes, `plane` doubles each), for the right-hand
// sides of [blockIdx.x * G, ...) that are still active.
__global__ void __launch_bounds__(TAIL_THREADS)
k_tail(TailParams P, const double* __restrict__ r_in, double* __restrict__ z_out, size_t plane, int B, int G,
       const int* __restrict__ active) {
    extern __shared__ __align__(16) double sm[];
    const int tid = threadIdx.x, ns = P.nlev - 1;  // ns smoothing levels
    // per level: hE, hS, s, sd, rh, ya, yb  -- each (ny+2) x (nx+2) with a zero border
    double *hE[TAIL_MAX_LEVELS], *hS[TAIL_MAX_LEVELS], *sS[TAIL_MAX_LEVELS], *sD[TAIL_MAX_LEVELS], *rh[TAIL_MAX_LEVELS],
        *ya[TAIL_MAX_LEVELS], *yb[TAIL_MAX_LEVELS];
    int W[TAIL_MAX_LEVELS];
    double* p = sm;
    for (int l = 0; l < ns; ++l) {
        const size_t S = (size_t)(P.lev[l].ny + 2) * (P.lev[l].nx + 2);
        W[l] = P.lev[l].nx + 2;
        hE[l] = p; hS[l] = p + S; sS[l] = p + 2 * S; sD[l] = p + 3 * S; rh[l] = p + 4 * S; ya[l] = p + 5 * S; yb[l] = p + 6 * S;
        p += 7 * S;
    }
    double* rc = p;        // coarsest right-hand side (<= 16)
    double* ecs = p + 16;  // coarsest correction
    double* pin = p + 32;  // its pseudo-inverse
    const Level& Lc = P.lev[ns];
    const int nc = Lc.ny * Lc.nx;
    // ---- resident data: zero everything (borders!), then the coefficients
    for (size_t i = tid; i < (size_t)(p - sm) + 32; i += TAIL_THREADS) sm[i] = 0.0;
    __syncthreads();
    for (int l = 0; l < ns; ++l) {
        const Level& L = P.lev[l];
        for (int i = tid; i < L.ny * L.nx; i += TAIL_THREADS) {
            const int y = i / L.nx, x = i % L.nx, g = y * L.pitch + x, s = (y + 1) * W[l] + x + 1;
            hE[l][s] = L.hE[g];
            hS[l][s] = L.hS[g];
            const float2 sc = L.sc[g];
            sS[l][s] = (double)sc.x;
            sD[l][s] = (double)sc.y;
        }
    }
    for (int i = tid; i < nc * nc; i += TAIL_THREADS) pin[i] = P.pinv[i];
    __syncthreads();

    const int b_end = min(B, (int)(blockIdx.x + 1) * G);
    for (int b = blockIdx.x * G; b < b_end; ++b) {
        if (active && !active[b]) continue;
        double* yc[TAIL_MAX_LEVELS];  // where the iterate of each level lives after its down sweeps
        // ---- level 0 right-hand side
        {
            const Level& L = P.lev[0];
            if (ns > 0) {
                for (int i = tid; i < L.ny * L.nx; i += TAIL_THREADS) {
                    const int y = i / L.nx, x = i % L.nx, s = (y + 1) * W[0] + x + 1;
                    rh[0][s] = sS[0][s] * r_in[b * plane + (size_t)y * L.pitch + x];
                }
            } else {
                for (int i = tid; i < nc; i += TAIL_THREADS) rc[i] = r_in[b * plane + (size_t)(i / L.nx) * L.pitch + i % L.nx];
            }
        }
        __syncthreads();
        // ---- down
        for (int l = 0; l < ns; ++l) {
            const Level& L = P.lev[l];
            const int n2 = L.ny * L.nx, w = W[l];
            double *cur = ya[l], *nxt = yb[l];
            for (int i = tid; i < n2; i += TAIL_THREADS) {
                const int s = (i / L.nx + 1) * w + i % L.nx + 1;
                cur[s] = P.ch.w[0] * rh[l][s];
            }
            __syncthreads();
            for (int k = 1; k < P.ch.nu; ++k) {
                const double wk = P.ch.w[k], a = 1.0 - wk;
                for (int i = tid; i < n2; i += TAIL_THREADS) {
                    const int s = (i / L.nx + 1) * w + i % L.nx + 1;
                    double t = fma(hE[l][s], cur[s + 1], rh[l][s]);
                    t = fma(hE[l][s - 1], cur[s - 1], t);
                    t = fma(hS[l][s], cur[s + w], t);
                    t = fma(hS[l][s - w], cur[s - w], t);
                    nxt[s] = fma(wk, t, a * cur[s]);
                }
                __syncthreads();
                double* tmp = cur; cur = nxt; nxt = tmp;
            }
            yc[l] = cur;
            // residual of the unscaled system, summed over 2x2 aggregates, into the next level
            const Level& Ln = P.lev[l + 1];
            const bool last = (l + 1 == ns);
            for (int i = tid; i < Ln.ny * Ln.nx; i += TAIL_THREADS) {
                const int Y = i / Ln.nx, X = i % Ln.nx;
                double v = 0.0;
#pragma unroll
                for (int dy = 0; dy < 2; ++dy)
#pragma unroll
                    for (int dx = 0; dx < 2; ++dx) {
                        const int fy = 2 * Y + dy, fx = 2 * X + dx;
                        if (fy < L.ny && fx < L.nx) {
                            const int s = (fy + 1) * w + fx + 1;
                            double t = fma(hE[l][s], cur[s + 1], rh[l][s]);
                            t = fma(hE[l][s - 1], cur[s - 1], t);
                            t = fma(hS[l][s], cur[s + w], t);
                            t = fma(hS[l][s - w], cur[s - w], t);
                            v = fma(sD[l][s], t - cur[s], v);
                        }
                    }
                if (last) rc[i] = v;
                else { const int s = (Y + 1) * W[l + 1] + X + 1; rh[l + 1][s] = sS[l + 1][s] * v; }
            }
            __syncthreads();
        }
        // ---- coarsest level: dense pseudo-inverse
        if (tid < nc) {
            double s = 0.0;
            for (int j = 0; j < nc; ++j) s = fma(pin[tid * nc + j], rc[j], s);
            ecs[tid] = s;
        }
        __syncthreads();
        // ---- up
        for (int l = ns - 1; l >= 0; --l) {
            const Level& L = P.lev[l];
            const Level& Ln = P.lev[l + 1];
            const int n2 = L.ny * L.nx, w = W[l];
            double* cur = yc[l];
            double* nxt = (cur == ya[l]) ? yb[l] : ya[l];
            const bool last = (l + 1 == ns);
            // correction of the coarser level (unscaled): ecs for the coarsest, else kept in that level's rh array
            for (int i = tid; i < n2; i += TAIL_THREADS) {
                const int y = i / L.nx, x = i % L.nx, s = (y + 1) * w + x + 1;
                const double e = last ? ecs[(y >> 1) * Ln.nx + (x >> 1)] : rh[l + 1][((y >> 1) + 1) * W[l + 1] + (x >> 1) + 1];
                cur[s] = fma(sD[l][s], e, cur[s]);
            }
            __syncthreads();
            for (int k = 0; k < P.ch.nu; ++k) {
                const double wk = P.ch.w[P.ch.nu - 1 - k], a = 1.0 - wk;
                for (int i = tid; i < n2; i += TAIL_THREADS) {
                    const int s = (i / L.nx + 1) * w + i % L.nx + 1;
                    double t = fma(hE[l][s], cur[s + 1], rh[l][s]);
                    t = fma(hE[l][s - 1], cur[s - 1], t);
                    t = fma(hS[l][s], cur[s + w], t);
                    t = fma(hS[l][s - w], cur[s - w], t);
                    nxt[s] = fma(wk, t, a * cur[s]);
                }
                __syncthreads();
                double* tmp = cur; cur = nxt; nxt = tmp;
            }
            // z = s y: to global memory on the tail's finest level, else into this level's rh array (the finer
            // level reads it as its coarse correction; rh is free now)
            for (int i = tid; i < n2; i += TAIL_THREADS) {
                const int y = i / L.nx, x = i % L.nx, s = (y + 1) * w + x + 1;
                const double z = sS[l][s] * cur[s];
                if (l == 0) z_out[b * plane + (size_t)y * L.pitch + x] = z;
                else rh[l][s] = z;
            }
            __syncthreads();
        }
        if (ns == 0) {  // the tail is the dense level alone
            const Level& L = P.lev[0];
            if (tid < nc) z_out[b * plane + (size_t)(tid / L.nx) * L.pitch + tid % L.nx] = ecs[tid];
            __syncthreads();
        }
    }
}

// acc[b] += sum over the nodes of a[b] * c[b]   (r.z on meshes whose level 0 is in the tail); grid.y = B.
// The pad column of an odd-width plane is skipped: k_tail never writes it, so it holds whatever the pool block
// held before (possibly a NaN bit pattern).
__global__ void __launch_bounds__(256)
k_dot_planes(const double* __restrict__ a, const double* __restrict__ c, size_t plane, int nx, int pitch,
             const int* __restrict__ active, double* __restrict__ acc) {
    __shared__ double red[32];
    const int b = blockIdx.y;
    if (active && !active[b]) return;
    double s = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < plane; i += (size_t)gridDim.x * blockDim.x)
        if ((int)(i % pitch) < nx) s = fma(a[b * plane + i], c[b * plane + i], s);
    s = block_sum(s, red);
    if (threadIdx.x == 0) atomicAdd(acc + b, s);
}

}  // namespace pdn
