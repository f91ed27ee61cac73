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
// grid = (tiles_x * tiles_y, ceil(B / GR)); block = GUESS_THREADS; a block keeps the raw conductances of its
// GUESS_TY x GUESS_TX tile in shared memory and loops over GR right-hand sides; per right-hand side it tabulates x0
// on the tile plus one ring (shared memory, double buffered: one __syncthreads per right-hand side) and applies
// the 5-point operator.
constexpr int GUESS_TX = 64, GUESS_TY = 16, GUESS_THREADS = 256;
__global__ void __launch_bounds__(GUESS_THREADS)
k_guess_rhs(GuessTable tab, Level L, const int* __restrict__ node, const int* __restrict__ src, double inv_n2,
            double* __restrict__ r0, double* __restrict__ rr0, double* __restrict__ sumx, int B, int GR) {
    constexpr int XW = GUESS_TX + 2, XH = GUESS_TY + 2;
    __shared__ double xs0[2][XH * XW];
    __shared__ double gE[GUESS_TY][GUESS_TX + 1];   // gE[y][x+1] = conductance (y, x)-(y, x+1); gE[y][0] = west of column 0
    __shared__ double gS[GUESS_TY + 1][GUESS_TX];   // gS[y+1][x] = conductance (y, x)-(y+1, x); gS[0][x] = north of row 0
    const int tiles_x = (L.nx + GUESS_TX - 1) / GUESS_TX;
    const int tx0 = (blockIdx.x % tiles_x) * GUESS_TX, ty0 = (blockIdx.x / tiles_x) * GUESS_TY;
    const int tid = threadIdx.x, lane = tid & 31;
    for (int i = tid; i < GUESS_TY * (GUESS_TX + 1); i += GUESS_THREADS) {
        const int y = ty0 + i / (GUESS_TX + 1), x = tx0 + i % (GUESS_TX + 1) - 1;
        gE[i / (GUESS_TX + 1)][i % (GUESS_TX + 1)] = (y < L.ny && x >= 0 && x < L.nx) ? L.gx[(size_t)y * L.pitch + x] : 0.0;
    }
    for (int i = tid; i < (GUESS_TY + 1) * GUESS_TX; i += GUESS_THREADS) {
        const int y = ty0 + i / GUESS_TX - 1, x = tx0 + i % GUESS_TX;
        gS[i / GUESS_TX][i % GUESS_TX] = (y >= 0 && y < L.ny && x < L.nx) ? L.gy[(size_t)y * L.pitch + x] : 0.0;
    }
    const size_t plane = (size_t)L.ny * L.pitch;
    const int b_end = min(B, (int)(blockIdx.y + 1) * GR);
    int buf = 0;
    for (int b = blockIdx.y * GR; b < b_end; ++b, buf ^= 1) {
        const int so = node[src[b]], ys = so / L.pitch, xs = so % L.pitch;
        double* xt = xs0[buf];
        for (int i = tid; i < XH * (XW / 2); i += GUESS_THREADS) {  // two neighbouring columns per step
            const int ry = i / (XW / 2), rx = 2 * (i % (XW / 2)), y = ty0 + ry - 1, x = tx0 + rx - 1;
            double v0 = 0.0, v1 = 0.0;
            if (y >= 0 && y < L.ny) {
                if (x >= 0 && x + 1 < L.nx) guess_x0_pair(tab, y, x, ys, xs, v0, v1);
                else {
                    if (x >= 0 && x < L.nx) v0 = guess_x0(tab, y, x, ys, xs);
                    if (x + 1 >= 0 && x + 1 < L.nx) v1 = guess_x0(tab, y, x + 1, ys, xs);
                }
            }
            xt[ry * XW + rx] = v0;
            xt[ry * XW + rx + 1] = v1;
        }
        __syncthreads();  // (also orders the coefficient tiles on the first pass)
        double rr = 0.0, sx = 0.0;
        for (int i = tid; i < GUESS_TY * GUESS_TX; i += GUESS_THREADS) {
            const int ly = i / GUESS_TX, lx = i % GUESS_TX, y = ty0 + ly, x = tx0 + lx;
            if (y >= L.ny || x >= L.pitch) continue;
            if (x >= L.nx) { r0[b * plane + (size_t)y * L.pitch + x] = 0.0; continue; }  // pad column of an odd-width plane
            const double c = xt[(ly + 1) * XW + lx + 1];
            const double e = gE[ly][lx + 1], w = gE[ly][lx], s = gS[ly + 1][lx], nn = gS[ly][lx];
            // (L x0)_i = sum over neighbours of g (x0_i - x0_nb); absent neighbours have g = 0
            double lx0 = e * (c - xt[(ly + 1) * XW + lx + 2]);
            lx0 = fma(w, c - xt[(ly + 1) * XW + lx], lx0);
            lx0 = fma(s, c - xt[(ly + 2) * XW + lx + 1], lx0);
            lx0 = fma(nn, c - xt[ly * XW + lx + 1], lx0);
            const double r = ((y == ys && x == xs) ? 1.0 - inv_n2 : -inv_n2) - lx0;
            r0[b * plane + (size_t)y * L.pitch + x] = r;
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
