// S1, initial guess of the port solves on a non-uniform tier (second half; PAPER.md:128
// "can be easily computed using Eq. (3)").
//
// BASELINE's tiers are a uniform mesh whose segments scatter around a mean (+-10 % jitter, 0.5 % of them removed).
// For the right-hand side b = e_src - 1/n^2 the mean mesh has the closed-form solution x0 = L_mean^+ b = column src
// of Wu's Eq. (3), which uniform.cuh tabulates: four look-ups per node.  PCG therefore starts from
//     x0,   r0 = b - L x0 = (L_mean - L) x0,      ||r0|| ~ 0.1 ||b||  on BASELINE's meshes,
// i.e. about one PCG iteration ahead, and the gathered port values are x0[port] + the PCG correction.  The guess
// only moves the starting point: the operator, the stopping test (||r|| <= rtol ||b||) and therefore the accuracy
// of the result are those of the plain solve, whatever the quality (or the FP32 storage) of the table -- provided
// the SAME x0 enters r0 and the gathered result, which is why both kernels below evaluate it through guess_x0().
// A right-hand side whose guess does not help (||r0|| > ||b|| / 2: a tier far from its mean mesh) falls back to
// x0 = 0 on the device (k_guess_check + k_init_rhs with the keep mask).
#pragma once
#include "common.cuh"
#include "uniform.cuh"

namespace pdn {

struct GuessTable {
    const float* G;   // table of (rho, 1), (n+1) x (n+1)
    const float2* P;  // the same values as pairs (G[t][s], G[t][s+1])
    double scale;     // 1 / mean g_y
    int n;
};

// columns a, b = a +- 1 of table row t with one 8-byte load
__device__ __forceinline__ void guess_pair(const GuessTable& t, int row, int a, int b, float& va, float& vb) {
    const float2 v = __ldg(t.P + (size_t)row * (t.n + 1) + min(a, b));
    va = a < b ? v.x : v.y;
    vb = a < b ? v.y : v.x;
}

// x0 at the two nodes (y, x) and (y, x + 1): bit-identical to guess_x0 of each (same values, same association)
__device__ __forceinline__ void guess_x0_pair(const GuessTable& t, int y, int x, int ys, int xs, double& v0, double& v1) {
    const int n = t.n, dy = abs(y - ys);
    int sy = y + ys + 1;
    sy = sy <= n ? sy : 2 * n - sy;
    const int dxa = abs(x - xs), dxb = abs(x + 1 - xs);
    int sxa = x + xs + 1, sxb = x + xs + 2;
    sxa = sxa <= n ? sxa : 2 * n - sxa;
    sxb = sxb <= n ? sxb : 2 * n - sxb;
    float ddA, ddB, dsA, dsB, sdA, sdB, ssA, ssB;  // G[dy][dx], G[dy][sx], G[sy][dx], G[sy][sx] at nodes A, B
    guess_pair(t, dy, dxa, dxb, ddA, ddB);
    guess_pair(t, dy, sxa, sxb, dsA, dsB);
    guess_pair(t, sy, dxa, dxb, sdA, sdB);
    guess_pair(t, sy, sxa, sxb, ssA, ssB);
    v0 = t.scale * (0.25 * (((double)ddA + (double)ssA) + ((double)dsA + (double)sdA)));
    v1 = t.scale * (0.25 * (((double)ddB + (double)ssB) + ((double)dsB + (double)sdB)));
}

__device__ __forceinline__ double guess_x0(const GuessTable& t, int y, int x, int ys, int xs) {
    return t.scale * spectral_entry<float>(t.G, t.n, y, x, ys, xs);
}

// r0[b] = b - L x0 on the pitched plane, rr0[b] += ||r0||^2, sumx[b] += sum(x0).
// grid = (tiles_x * tiles_y, ceil(B / GR)); block = GUESS_THREADS; a thread keeps the raw conductances of its four
// nodes of the GUESS_TY x GUESS_TX tile in registers and loops over GR right-hand sides; per right-hand side the block
// tabulates x0 on the tile plus one ring (shared memory, double buffered: one __syncthreads per right-hand side) and
// applies the 5-point operator.  Everything that does not depend on the right-hand side (which table entries a
// thread evaluates, its nodes, their coefficients) is set up once per block: the kernel is instruction-bound.
constexpr int GUESS_TX = 64, GUESS_TY = 16, GUESS_THREADS = 256;
__global__ void __launch_bounds__(GUESS_THREADS)
k_guess_rhs(GuessTable tab, Level L, const int* __restrict__ node, const int* __restrict__ src, double inv_n2,
            double* __restrict__ r0, double* __restrict__ rr0, double* __restrict__ sumx, int B, int GR) {
    constexpr int XW = GUESS_TX + 2, XH = GUESS_TY + 2, NPAIR = XH * (XW / 2);
    constexpr int PER = (NPAIR + GUESS_THREADS - 1) / GUESS_THREADS;       // pair entries of the ring tile per thread
    constexpr int NODES = GUESS_TY * GUESS_TX / GUESS_THREADS;             // tile nodes per thread (same column)
    static_assert(GUESS_THREADS % GUESS_TX == 0 && (GUESS_TY * GUESS_TX) % GUESS_THREADS == 0, "tile / block shape");
    __shared__ __align__(16) double xs0[2][XH * XW];
    const int tiles_x = (L.nx + GUESS_TX - 1) / GUESS_TX;
    const int tx0 = (blockIdx.x % tiles_x) * GUESS_TX, ty0 = (blockIdx.x / tiles_x) * GUESS_TY;
    const int tid = threadIdx.x, lane = tid & 31;
    // ---- per-thread constants of the tabulation: entry k covers ring-tile columns rx, rx+1 of ring-tile row ry
    int ey[PER], ex[PER], eo[PER], ekind[PER];  // mesh row, mesh column of the first node, offset in xs0, 0 none / 1 pair / 2 singles
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int i = tid + k * GUESS_THREADS, ry = i / (XW / 2), rx = 2 * (i % (XW / 2));
        ey[k] = ty0 + ry - 1; ex[k] = tx0 + rx - 1; eo[k] = ry * XW + rx;
        const bool row_ok = i < NPAIR && ey[k] >= 0 && ey[k] < L.ny;
        ekind[k] = i >= NPAIR ? -1 : !row_ok ? 0 : (ex[k] >= 0 && ex[k] + 1 < L.nx) ? 1 : 2;
    }
    // ---- per-thread constants of the operator: nodes (ly0 + k * step, lx), their four conductances
    const int lx = tid % GUESS_TX, ly0 = tid / GUESS_TX, x = tx0 + lx;
    constexpr int STEP = GUESS_THREADS / GUESS_TX;
    double ge[NODES], gw[NODES], gs[NODES], gn[NODES];
    int nkind[NODES];  // 0 outside the plane, 1 node, 2 pad column
#pragma unroll
    for (int k = 0; k < NODES; ++k) {
        const int y = ty0 + ly0 + k * STEP;
        nkind[k] = (y >= L.ny || x >= L.pitch) ? 0 : x >= L.nx ? 2 : 1;
        const bool in = nkind[k] == 1;
        const size_t o = (size_t)y * L.pitch + x;
        ge[k] = in ? L.gx[o] : 0.0;                       // pad / last column of gx is zero
        gw[k] = (in && x > 0) ? L.gx[o - 1] : 0.0;
        gs[k] = in ? L.gy[o] : 0.0;                       // last row of gy is zero
        gn[k] = (in && y > 0) ? L.gy[o - L.pitch] : 0.0;
    }
    const size_t plane = (size_t)L.ny * L.pitch;
    const int b_end = min(B, (int)(blockIdx.y + 1) * GR);
    int buf = 0;
    for (int b = blockIdx.y * GR; b < b_end; ++b, buf ^= 1) {
        const int so = node[src[b]], ys = so / L.pitch, xs = so % L.pitch;
        double* xt = xs0[buf];
#pragma unroll
        for (int k = 0; k < PER; ++k) {
            if (ekind[k] < 0) continue;
            double v0 = 0.0, v1 = 0.0;
            if (ekind[k] == 1) guess_x0_pair(tab, ey[k], ex[k], ys, xs, v0, v1);
            else if (ekind[k] == 2) {
                if (ex[k] >= 0 && ex[k] < L.nx) v0 = guess_x0(tab, ey[k], ex[k], ys, xs);
                if (ex[k] + 1 >= 0 && ex[k] + 1 < L.nx) v1 = guess_x0(tab, ey[k], ex[k] + 1, ys, xs);
            }
            *reinterpret_cast<double2*>(xt + eo[k]) = make_double2(v0, v1);  // eo is even, XW is even
        }
        __syncthreads();
        double rr = 0.0, sx = 0.0;
        double* rp = r0 + b * plane + (size_t)(ty0 + ly0) * L.pitch + x;
#pragma unroll
        for (int k = 0; k < NODES; ++k, rp += (size_t)STEP * L.pitch) {
            if (nkind[k] == 0) continue;
            if (nkind[k] == 2) { *rp = 0.0; continue; }  // pad column of an odd-width plane
            const int ly = ly0 + k * STEP;
            const double* xc = xt + (ly + 1) * XW + lx + 1;
            const double c = xc[0];
            // (L x0)_i = sum over neighbours of g (x0_i - x0_nb); absent neighbours have g = 0
            double lx0 = ge[k] * (c - xc[1]);
            lx0 = fma(gw[k], c - xc[-1], lx0);
            lx0 = fma(gs[k], c - xc[XW], lx0);
            lx0 = fma(gn[k], c - xc[-XW], lx0);
            const double r = ((ty0 + ly == ys && x == xs) ? 1.0 - inv_n2 : -inv_n2) - lx0;
            *rp = r;
            rr = fma(r, r, rr);
            sx += c;
        }
        rr = warp_sum(rr);
        sx = warp_sum(sx);
        if (lane == 0) { atomicAdd(rr0 + b, rr); atomicAdd(sumx + b, sx); }  // one atomic per warp and quantity
    }
}

// Terminal-source solves deliver ONE number, Z[s,s] = b^T L^+ b, and stop early because the CG error of b^T x_k is the
// SQUARE of the energy-norm error -- but only when x_0 = 0: from a guess, b^T (x - x_k) = e_k^T L x_0 + e_k^T L e_k is
// first order again.  The energy form of the same number, 2 b^T x_k - x_k^T L x_k = b^T x_k + x_k^T r_k, is second
// order from any starting point, and CG makes x_k - x_0 orthogonal to r_k, so the correction is the single dot
//     dot[b] = x_0^T r_k      (x_0 re-evaluated from the table; r_k = the right-hand side's last residual),
// added to x_k[s] - mean(x_k) by k_finish_term.  r_k lives in the ping-pong buffer that was current when the
// right-hand side converged (rbuf_of[b], recorded by k_scal_check).  grid = (tiles, B), 64 x 64 nodes per block.
constexpr int GDOT_T = 64;
__global__ void __launch_bounds__(256)
k_guess_dot(GuessTable tab, int ny, int nx, int pitch, size_t plane, const int* __restrict__ node, const int* __restrict__ src,
            const int* __restrict__ keep, const double* __restrict__ ra, const double* __restrict__ rb,
            const int* __restrict__ rbuf_of, double* __restrict__ dot) {
    const int b = blockIdx.y;
    if (!keep[b]) return;
    const int tiles_x = (nx + GDOT_T - 1) / GDOT_T;
    const int tx0 = (blockIdx.x % tiles_x) * GDOT_T, ty0 = (blockIdx.x / tiles_x) * GDOT_T;
    const double* r = (rbuf_of[b] ? rb : ra) + b * plane;
    const int so = node[src[b]], ys = so / pitch, xs = so % pitch;
    double s = 0.0;
    for (int i = threadIdx.x; i < GDOT_T * (GDOT_T / 2); i += 256) {  // two neighbouring columns per step
        const int y = ty0 + i / (GDOT_T / 2), x = tx0 + 2 * (i % (GDOT_T / 2));
        if (y >= ny || x >= nx) continue;
        if (x + 1 < nx) {
            double v0, v1;
            guess_x0_pair(tab, y, x, ys, xs, v0, v1);
            const double2 rv = *reinterpret_cast<const double2*>(r + (size_t)y * pitch + x);  // x and pitch are even
            s = fma(v0, rv.x, s);
            s = fma(v1, rv.y, s);
        } else {
            s = fma(guess_x0(tab, y, x, ys, xs), r[(size_t)y * pitch + x], s);
        }
    }
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) atomicAdd(dot + b, s);
}

// keep[b] = 1 if the guess of right-hand side b is used (it at least halves the residual), else 0
__global__ void k_guess_check(const double* __restrict__ rr0, double bnorm2, int* __restrict__ keep, int B) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < B) keep[b] = rr0[b] <= 0.25 * bnorm2 ? 1 : 0;
}

// Starting values of the accumulators the PCG loop adds to: the gathered port values
//   xport[b][k] = x0_b[node k]  (TSV-source batch, k over the tier's ports)  /  xown[b] = x0_b[its own node]
// and the mean of x0 (xmean[b]); zero for a right-hand side whose guess was rejected.  grid = (ceil(max(ngather,1)/128), B)
__global__ void k_guess_ports(GuessTable tab, int pitch, const int* __restrict__ node, int ngather, const int* __restrict__ src,
                              const int* __restrict__ keep, const double* __restrict__ sumx, double inv_n2,
                              double* __restrict__ xport, double* __restrict__ xown, double* __restrict__ xmean, int B) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    const bool use = keep[b] != 0;
    const int so = node[src[b]], ys = so / pitch, xs = so % pitch;
    if (ngather > 0) {
        if (k < ngather) {
            const int o = node[k];
            xport[(size_t)b * ngather + k] = use ? guess_x0(tab, o / pitch, o % pitch, ys, xs) : 0.0;
        }
    } else if (k == 0) {
        xown[b] = use ? guess_x0(tab, ys, xs, ys, xs) : 0.0;
    }
    if (k == 0) xmean[b] = use ? sumx[b] * inv_n2 : 0.0;
}

}  // namespace pdn
