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

// The four look-ups of Eq. (3) are summed in FP32, in one fixed order (explicitly rounded operations: no contraction),
// and converted once: FP32 -> FP64 conversions run on the SM's conversion pipe, and four per node made it the busiest
// unit of the guess kernels.  A guess needs no more than FP32; what matters is that every kernel gets the same bits.
__device__ __forceinline__ float guess_sum4(float dd, float ss, float ds, float sd) {
    return __fmul_rn(0.25f, __fadd_rn(__fadd_rn(dd, ss), __fadd_rn(ds, sd)));
}

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
    v0 = t.scale * (double)guess_sum4(ddA, ssA, dsA, sdA);
    v1 = t.scale * (double)guess_sum4(ddB, ssB, dsB, sdB);
}

__device__ __forceinline__ double guess_x0(const GuessTable& t, int y, int x, int ys, int xs) {
    const int n = t.n, dx = abs(x - xs), dy = abs(y - ys);
    int sx = x + xs + 1, sy = y + ys + 1;
    sx = sx <= n ? sx : 2 * n - sx;
    sy = sy <= n ? sy : 2 * n - sy;
    const size_t ld = (size_t)n + 1;
    return t.scale * (double)guess_sum4(__ldg(t.G + dy * ld + dx), __ldg(t.G + sy * ld + sx), __ldg(t.G + dy * ld + sx), __ldg(t.G + sy * ld + dx));
}

// r0[b] = b - L x0 on the pitched plane, rr0[b] += ||r0||^2, sumx[b] += sum(x0).
// grid = (tiles_x * tiles_y, ceil(B / GR)); block = GUESS_THREADS; a thread owns a 2 x 2 patch of the GUESS_TY x
// GUESS_TX tile (its conductances in registers) and loops over GR right-hand sides; per right-hand side the block
// tabulates x0 on the tile plus one ring (shared memory, double buffered: one __syncthreads per right-hand side;
// mesh column j of the tile sits at index j + 2 of a 68-wide row, so that column pairs are 16-byte aligned) and
// applies the 5-point operator with 16-byte shared loads and global stores.  Everything that does not depend on
// the right-hand side is set up once per block.
constexpr int GUESS_TX = 64, GUESS_TY = 16, GUESS_THREADS = 256;
__global__ void __launch_bounds__(GUESS_THREADS)
k_guess_rhs(GuessTable tab, Level L, const int* __restrict__ node, const int* __restrict__ src, double inv_n2,
            double* __restrict__ r0, double* __restrict__ rr0, double* __restrict__ sumx, int B, int GR) {
    constexpr int XW = GUESS_TX + 4, XH = GUESS_TY + 2, EPR = GUESS_TX / 2 + 2, NENT = XH * EPR;  // entries per ring row: 32 pairs + 2 singles
    constexpr int PER = (NENT + GUESS_THREADS - 1) / GUESS_THREADS;
    static_assert((GUESS_TX / 2) * (GUESS_TY / 2) == GUESS_THREADS, "one 2 x 2 patch per thread");
    __shared__ __align__(16) double xs0[2][XH * XW];
    __shared__ double part[2][2][GUESS_THREADS / 32];  // per-warp partial sums of the two reductions, double buffered
    const int tiles_x = (L.nx + GUESS_TX - 1) / GUESS_TX;
    const int tx0 = (blockIdx.x % tiles_x) * GUESS_TX, ty0 = (blockIdx.x / tiles_x) * GUESS_TY;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // the block's partial sums of right-hand side b go out as ONE atomic per quantity (1024 blocks add to the same two
    // words per right-hand side: per-warp atomics were the kernel's bottleneck), one iteration later: after the next
    // __syncthreads the eight per-warp values are visible to threads 0 and 1
    auto flush = [&](int bb, int pb) {
        if (tid < 2) {
            double v = 0.0;
#pragma unroll
            for (int w = 0; w < GUESS_THREADS / 32; ++w) v += part[pb][tid][w];
            atomicAdd((tid == 0 ? rr0 : sumx) + bb, v);
        }
    };
    // ---- per-thread constants of the tabulation
    int ey[PER], ex[PER], eo[PER], ekind[PER];  // mesh row, first mesh column, offset in xs0; -1 nothing, 0 zeros, 1 pair, 2 first only, 3 single
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int i = tid + k * GUESS_THREADS, ry = i / EPR, e = i % EPR;
        ey[k] = ty0 + ry - 1;
        const bool row_ok = ey[k] >= 0 && ey[k] < L.ny;
        if (e < GUESS_TX / 2) {  // columns 2e, 2e+1 of the tile
            ex[k] = tx0 + 2 * e; eo[k] = ry * XW + 2 * e + 2;
            ekind[k] = i >= NENT ? -1 : (!row_ok || ex[k] >= L.nx) ? 0 : ex[k] + 1 < L.nx ? 1 : 2;
        } else {                 // ring column -1 (e == 32) or GUESS_TX (e == 33)
            const int j = e == GUESS_TX / 2 ? -1 : GUESS_TX;
            ex[k] = tx0 + j; eo[k] = ry * XW + j + 2;
            ekind[k] = i >= NENT ? -1 : (row_ok && ex[k] >= 0 && ex[k] < L.nx) ? 3 : 4;  // 4: a single zero
        }
    }
    // ---- per-thread constants of the operator: patch rows 2 pr, 2 pr + 1, columns 2 pc, 2 pc + 1
    const int pc = tid % (GUESS_TX / 2), pr = tid / (GUESS_TX / 2), x = tx0 + 2 * pc, y = ty0 + 2 * pr;
    double ge[2][2], gw[2], gs[2][2], gn[2];  // east of both columns, west of column 0; south of both rows, north of row 0
    bool in[2][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            in[i][j] = y + i < L.ny && x + j < L.nx;
            const size_t o = (size_t)(y + i) * L.pitch + x + j;
            ge[i][j] = in[i][j] ? L.gx[o] : 0.0;   // (zero in the last column of the mesh)
            gs[i][j] = in[i][j] ? L.gy[o] : 0.0;   // (zero in the last row)
        }
#pragma unroll
    for (int i = 0; i < 2; ++i) gw[i] = (in[i][0] && x > 0) ? L.gx[(size_t)(y + i) * L.pitch + x - 1] : 0.0;
#pragma unroll
    for (int j = 0; j < 2; ++j) gn[j] = (in[0][j] && y > 0) ? L.gy[(size_t)(y - 1) * L.pitch + x + j] : 0.0;
    const bool row_in[2] = {y < L.ny && x < L.pitch, y + 1 < L.ny && x < L.pitch};  // x even: both columns are addressable
    const size_t plane = (size_t)L.ny * L.pitch;
    const int b_end = min(B, (int)(blockIdx.y + 1) * GR);
    int buf = 0;
    for (int b = blockIdx.y * GR; b < b_end; ++b, buf ^= 1) {
        const int so = node[src[b]], ys = so / L.pitch, xs = so % L.pitch;
        double* xt = xs0[buf];
#pragma unroll
        for (int k = 0; k < PER; ++k) {
            if (ekind[k] < 0) continue;
            if (ekind[k] >= 3) { xt[eo[k]] = ekind[k] == 3 ? guess_x0(tab, ey[k], ex[k], ys, xs) : 0.0; continue; }
            double v0 = 0.0, v1 = 0.0;
            if (ekind[k] == 1) guess_x0_pair(tab, ey[k], ex[k], ys, xs, v0, v1);
            else if (ekind[k] == 2) v0 = guess_x0(tab, ey[k], ex[k], ys, xs);
            *reinterpret_cast<double2*>(xt + eo[k]) = make_double2(v0, v1);
        }
        __syncthreads();
        if (b > (int)blockIdx.y * GR) flush(b - 1, buf ^ 1);
        // rows 2 pr - 1 .. 2 pr + 2 of the ring tile (ring row = tile row + 1), columns 2 pc, 2 pc + 1 (+ the two beside them)
        const double* xc = xt + (2 * pr) * XW + 2 * pc + 2;
        const double2 up = *reinterpret_cast<const double2*>(xc), c0 = *reinterpret_cast<const double2*>(xc + XW),
                      c1 = *reinterpret_cast<const double2*>(xc + 2 * XW), dn = *reinterpret_cast<const double2*>(xc + 3 * XW);
        const double w0 = xc[XW - 1], e0 = xc[XW + 2], w1 = xc[2 * XW - 1], e1 = xc[2 * XW + 2];
        // (L x0)_i = sum over neighbours of g (x0_i - x0_nb); absent neighbours have g = 0
        double l00 = ge[0][0] * (c0.x - c0.y), l01 = ge[0][1] * (c0.y - e0);
        l00 = fma(gw[0], c0.x - w0, l00);       l01 = fma(ge[0][0], c0.y - c0.x, l01);
        l00 = fma(gs[0][0], c0.x - c1.x, l00);  l01 = fma(gs[0][1], c0.y - c1.y, l01);
        l00 = fma(gn[0], c0.x - up.x, l00);     l01 = fma(gn[1], c0.y - up.y, l01);
        double l10 = ge[1][0] * (c1.x - c1.y), l11 = ge[1][1] * (c1.y - e1);
        l10 = fma(gw[1], c1.x - w1, l10);       l11 = fma(ge[1][0], c1.y - c1.x, l11);
        l10 = fma(gs[1][0], c1.x - dn.x, l10);  l11 = fma(gs[1][1], c1.y - dn.y, l11);
        l10 = fma(gs[0][0], c1.x - c0.x, l10);  l11 = fma(gs[0][1], c1.y - c0.y, l11);
        const bool sy0 = y == ys, sy1 = y + 1 == ys, sx0 = x == xs, sx1 = x + 1 == xs;
        // pad entries (the pad column of an odd-width plane) are written as zeros
        const double r00 = in[0][0] ? ((sy0 && sx0) ? 1.0 - inv_n2 : -inv_n2) - l00 : 0.0;
        const double r01 = in[0][1] ? ((sy0 && sx1) ? 1.0 - inv_n2 : -inv_n2) - l01 : 0.0;
        const double r10 = in[1][0] ? ((sy1 && sx0) ? 1.0 - inv_n2 : -inv_n2) - l10 : 0.0;
        const double r11 = in[1][1] ? ((sy1 && sx1) ? 1.0 - inv_n2 : -inv_n2) - l11 : 0.0;
        double* rp = r0 + b * plane + (size_t)y * L.pitch + x;
        if (row_in[0]) *reinterpret_cast<double2*>(rp) = make_double2(r00, r01);
        if (row_in[1]) *reinterpret_cast<double2*>(rp + L.pitch) = make_double2(r10, r11);
        double rr = fma(r00, r00, fma(r01, r01, fma(r10, r10, r11 * r11)));
        double sx = (in[0][0] ? c0.x : 0.0) + (in[0][1] ? c0.y : 0.0) + (in[1][0] ? c1.x : 0.0) + (in[1][1] ? c1.y : 0.0);
        rr = warp_sum(rr);
        sx = warp_sum(sx);
        if (lane == 0) { part[buf][0][warp] = rr; part[buf][1][warp] = sx; }
    }
    __syncthreads();
    if (b_end > (int)blockIdx.y * GR) flush(b_end - 1, buf ^ 1);
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
