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
// the SAME x0 enters r0 and the gathered result: k_guess_rhs sums the same four FP32 values in the order of guess_x0().
// A right-hand side whose guess does not help (||r0|| > ||b|| / 2: a tier far from its mean mesh) falls back to
// x0 = 0 on the device (k_guess_check + k_init_rhs with the keep mask).
#pragma once
#include "common.cuh"
#include "stencil3.cuh"
#include "uniform.cuh"

namespace pdn {

struct GuessTable {
    const float* G;   // table of (rho, 1), (n+1) x (n+1)
    double scale;     // 1 / mean g_y
    int n;
};

// The four look-ups of Eq. (3) are summed in FP32, in one fixed order (explicitly rounded operations: no contraction),
// and converted once: FP32 -> FP64 conversions run on the SM's conversion pipe, and four per node made it the busiest
// unit of the guess kernels.  A guess needs no more than FP32; what matters is that every kernel gets the same bits.
__device__ __forceinline__ float guess_sum4(float dd, float ss, float ds, float sd) {
    return __fmul_rn(0.25f, __fadd_rn(__fadd_rn(dd, ss), __fadd_rn(ds, sd)));
}

__device__ __forceinline__ double guess_x0(const GuessTable& t, int y, int x, int ys, int xs) {
    const int n = t.n, dx = abs(x - xs), dy = abs(y - ys);
    int sx = x + xs + 1, sy = y + ys + 1;
    sx = sx <= n ? sx : 2 * n - sx;
    sy = sy <= n ? sy : 2 * n - sy;
    const size_t ld = (size_t)n + 1;
    return t.scale * (double)guess_sum4(__ldg(t.G + dy * ld + dx), __ldg(t.G + sy * ld + sx), __ldg(t.G + dy * ld + sx), __ldg(t.G + sy * ld + dx));
}

// r0[b] = b - L x0 on the pitched plane, rr0[b] += ||r0||^2, sumx[b] += sum(x0), xr0[b] += x0 . r0.
//
// The table windows are staged by TMA.  For one right-hand side (source column xs, row ys) the nodes of a tile of
// 64 x TY mesh nodes plus its ring use, in each of the four index combinations, a CONTIGUOUS window of at most
// (TY + 2) x 66 table entries: over consecutive x the difference index |x - xs| runs down to 0 left of the source and
// up again right of it, and the folded sum index f(x + xs + 1) runs up to n and back down -- a run or a V, never a
// gap.  So the block asks the TMA unit for four 2D boxes of the table (origin = the smallest index the tile uses,
// guess_origin) per right-hand side, NST stages ahead, and its threads read them with 4-byte shared loads at
// row * 72 + column -- forwards or backwards; a lane's two columns make the warp's addresses 8 bytes apart, a two-way
// bank conflict at worst -- instead of gathering sixteen bytes per node from L2 through the L1TEX path (round 2's
// first version: 7 us per right-hand side at 1024^2, L1TEX-bound; this one 4.1 us, bound by instruction issue and
// latency at 16 warps per SM: ablating the TMA fetches or the stores changes nothing).
// The innermost box coordinate has to be a multiple of 16 bytes (an odd one is an illegal instruction), so the column
// origin is rounded down to a multiple of four entries and the box is 72 wide: 66 entries used, up to 3 skipped.
// grid = (tiles_x * tiles_y, ceil(B / GR)); block = W warps; lane l of warp w owns columns 2l, 2l+1 and rows
// R w .. R w + R - 1 of the tile with its conductances in registers, evaluates x0 on those rows and the two beside
// them, gets the columns beside its own from the neighbouring lanes (lanes 0 and 31 look their ring column up) and
// applies the 5-point operator.  One __syncthreads per right-hand side (stage consumed -> refill).
constexpr int GW_TX = 64, GW_BW = 72, GW_MAX_GR = 64;

__device__ __forceinline__ int guess_fold(int t, int n) { return t <= n ? t : 2 * n - t; }

// smallest |x - s| (a_d) and smallest f(x + s + 1) (a_s) over the mesh coordinates x in [lo, hi]
__device__ __forceinline__ void guess_origin(int lo, int hi, int s, int n, int& a_d, int& a_s) {
    a_d = max(max(lo - s, s - hi), 0);
    const int tlo = lo + s + 1, thi = hi + s + 1;
    a_s = thi <= n ? tlo : (tlo > n ? 2 * n - thi : min(tlo, 2 * n - thi));
}

template <int R, int W>
struct GuessGeom {
    static constexpr int TY = R * W, BH = TY + 2;
    static constexpr int WIN = (BH * GW_BW + 31) & ~31;  // floats per window, a multiple of 128 bytes (TMA destination)
    static constexpr uint32_t BOX_BYTES = BH * GW_BW * sizeof(float);
    static constexpr size_t STAGE_BYTES = 4 * (size_t)WIN * sizeof(float);
};

template <int R, int W, int NST>
__global__ void __launch_bounds__(32 * W)
k_guess_rhs(const __grid_constant__ CUtensorMap tm_tab, double scale, Level L, const int* __restrict__ node,
            const int* __restrict__ src, double inv_n2, double* __restrict__ r0, double* __restrict__ rr0,
            double* __restrict__ sumx, double* __restrict__ xr0, int B, int GR) {
    using Gm = GuessGeom<R, W>;
    constexpr int TY = Gm::TY, WIN = Gm::WIN;
    extern __shared__ __align__(128) float win[];  // NST stages x 4 windows: (dy,dx) (sy,sx) (dy,sx) (sy,dx)
    __shared__ uint64_t mbar[NST];
    __shared__ int s_xs[GW_MAX_GR], s_ys[GW_MAX_GR];
    __shared__ double part[2][3][W];  // per-warp partial sums of the three reductions, double buffered
    const int n = L.nx;               // tiers are square: the table is (n + 1) x (n + 1)
    const int tiles_x = (L.nx + GW_TX - 1) / GW_TX;
    const int tx0 = (blockIdx.x % tiles_x) * GW_TX, ty0 = (blockIdx.x / tiles_x) * TY;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b0 = blockIdx.y * GR, nb = min(GR, B - b0);
    for (int j = tid; j < nb; j += 32 * W) {
        const int so = node[src[b0 + j]];
        s_ys[j] = so / L.pitch;
        s_xs[j] = so % L.pitch;
    }
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(&mbar[s], 1);
        mbar_fence_init();
    }
    // mesh coordinates the tile and its ring use (clamped to the mesh: what lies outside is never multiplied by a
    // non-zero conductance, but its index has to stay inside the window)
    const int xlo = max(tx0 - 1, 0), xhi = min(tx0 + GW_TX, L.nx - 1);
    const int ylo = max(ty0 - 1, 0), yhi = min(ty0 + TY, L.ny - 1);
    // ---- per-thread constants of the operator
    const int x = tx0 + 2 * lane, y = ty0 + R * warp;
    double ge0[R], ge1[R], gw[R], gs0[R], gs1[R], gn0 = 0.0, gn1 = 0.0;  // east of both columns, west of column 0, south
    unsigned in0 = 0, in1 = 0, rowin = 0;  // bit i: node (y + i, x) / (y + i, x + 1) is a mesh node; the row pair is addressable
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const int yy = y + i;
        const bool ok = yy < L.ny && x < L.pitch;  // x and pitch are even: both columns are addressable (pads hold zeros)
        const size_t o = (size_t)yy * L.pitch + x;
        const double2 e = ok ? ldg2(L.gx + o) : make_double2(0.0, 0.0);
        const double2 s = ok ? ldg2(L.gy + o) : make_double2(0.0, 0.0);
        ge0[i] = e.x; ge1[i] = e.y; gs0[i] = s.x; gs1[i] = s.y;
        gw[i] = (ok && x > 0) ? __ldg(L.gx + o - 1) : 0.0;
        if (ok) rowin |= 1u << i;
        if (ok && x < L.nx) in0 |= 1u << i;
        if (ok && x + 1 < L.nx) in1 |= 1u << i;
    }
    if (y > 0 && y - 1 < L.ny && x < L.pitch) {
        const double2 s = ldg2(L.gy + (size_t)(y - 1) * L.pitch + x);
        gn0 = s.x; gn1 = s.y;
    }
    const int xc0 = min(x, n - 1), xc1 = min(x + 1, n - 1);
    const bool edge = lane == 0 || lane == 31;
    const int xce = lane == 0 ? max(x - 1, 0) : min(x + 2, n - 1);  // the ring column of lanes 0 / 31
    const size_t plane = (size_t)L.ny * L.pitch;
    __syncthreads();
    auto fetch = [&](int j) {  // thread 0 only
        const int st = j % NST;
        float* w = win + (size_t)st * 4 * WIN;
        int adx, asx, ady, asy;
        guess_origin(xlo, xhi, s_xs[j], n, adx, asx);
        guess_origin(ylo, yhi, s_ys[j], n, ady, asy);
        adx &= ~3; asx &= ~3;
        mbar_expect_tx(&mbar[st], 4 * Gm::BOX_BYTES);
        tma_load_2d(w, &tm_tab, adx, ady, &mbar[st]);
        tma_load_2d(w + WIN, &tm_tab, asx, asy, &mbar[st]);
        tma_load_2d(w + 2 * WIN, &tm_tab, asx, ady, &mbar[st]);
        tma_load_2d(w + 3 * WIN, &tm_tab, adx, asy, &mbar[st]);
    };
    if (tid == 0)
        for (int j = 0; j < NST && j < nb; ++j) fetch(j);
    // the block's partial sums of right-hand side b go out as ONE atomic per quantity, one iteration later: after the
    // next __syncthreads the per-warp values are visible to threads 0 .. 2
    auto flush = [&](int bb, int pb) {
        if (tid < 3) {
            double v = 0.0;
#pragma unroll
            for (int w = 0; w < W; ++w) v += part[pb][tid][w];
            atomicAdd((tid == 0 ? rr0 : tid == 1 ? sumx : xr0) + bb, v);
        }
    };
    for (int j = 0; j < nb; ++j) {
        const int b = b0 + j, st = j % NST, buf = j & 1;
        const int xs = s_xs[j], ys = s_ys[j];
        int adx, asx, ady, asy;
        guess_origin(xlo, xhi, xs, n, adx, asx);
        guess_origin(ylo, yhi, ys, n, ady, asy);
        adx &= ~3; asx &= ~3;
        const int cd0 = abs(xc0 - xs) - adx, cd1 = abs(xc1 - xs) - adx, cde = abs(xce - xs) - adx;
        const int cs0 = guess_fold(xc0 + xs + 1, n) - asx, cs1 = guess_fold(xc1 + xs + 1, n) - asx, cse = guess_fold(xce + xs + 1, n) - asx;
        const float* wdd = win + (size_t)st * 4 * WIN;
        const float *wss = wdd + WIN, *wds = wdd + 2 * WIN, *wsd = wdd + 3 * WIN;
        mbar_wait(&mbar[st], (j / NST) & 1);
        float f0[R + 2], f1[R + 2], fe[R];  // rows y - 1 .. y + R of the two columns; rows y .. y + R - 1 of the ring column
#pragma unroll
        for (int i = 0; i < R + 2; ++i) {
            const int yy = min(max(y - 1 + i, 0), L.ny - 1);
            const int rd = (abs(yy - ys) - ady) * GW_BW, rs = (guess_fold(yy + ys + 1, n) - asy) * GW_BW;
            f0[i] = guess_sum4(wdd[rd + cd0], wss[rs + cs0], wds[rd + cs0], wsd[rs + cd0]);
            f1[i] = guess_sum4(wdd[rd + cd1], wss[rs + cs1], wds[rd + cs1], wsd[rs + cd1]);
            if (i >= 1 && i <= R && edge) fe[i - 1] = guess_sum4(wdd[rd + cde], wss[rs + cse], wds[rd + cse], wsd[rs + cde]);
        }
        __syncthreads();  // the stage is consumed; the partial sums of the previous right-hand side are visible
        if (tid == 0 && j + NST < nb) fetch(j + NST);
        if (j > 0) flush(b - 1, buf ^ 1);
        double v0[R + 2], v1[R + 2];
#pragma unroll
        for (int i = 0; i < R + 2; ++i) {
            v0[i] = scale * (double)f0[i];
            v1[i] = scale * (double)f1[i];
        }
        double rr = 0.0, sx = 0.0, xr = 0.0;
        double* rp = r0 + b * plane + (size_t)y * L.pitch + x;
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double c0 = v0[i + 1], c1 = v1[i + 1];
            double wl = __shfl_up_sync(0xffffffffu, c1, 1), er = __shfl_down_sync(0xffffffffu, c0, 1);
            if (edge) {
                const double ve = scale * (double)fe[i];
                if (lane == 0) wl = ve; else er = ve;
            }
            const double n0 = i == 0 ? gn0 : gs0[i == 0 ? 0 : i - 1], n1 = i == 0 ? gn1 : gs1[i == 0 ? 0 : i - 1];
            // (L x0)_i = sum over neighbours of g (x0_i - x0_nb); absent neighbours have g = 0
            double l0 = ge0[i] * (c0 - c1), l1 = ge1[i] * (c1 - er);
            l0 = fma(gw[i], c0 - wl, l0);          l1 = fma(ge0[i], c1 - c0, l1);
            l0 = fma(gs0[i], c0 - v0[i + 2], l0);  l1 = fma(gs1[i], c1 - v1[i + 2], l1);
            l0 = fma(n0, c0 - v0[i], l0);          l1 = fma(n1, c1 - v1[i], l1);
            const bool a0 = (in0 >> i) & 1, a1 = (in1 >> i) & 1, sy = y + i == ys;
            // pad entries (the pad column of an odd-width plane) are written as zeros
            const double q0 = a0 ? ((sy && x == xs) ? 1.0 - inv_n2 : -inv_n2) - l0 : 0.0;
            const double q1 = a1 ? ((sy && x + 1 == xs) ? 1.0 - inv_n2 : -inv_n2) - l1 : 0.0;
            if ((rowin >> i) & 1) *reinterpret_cast<double2*>(rp) = make_double2(q0, q1);
            rp += L.pitch;
            rr = fma(q0, q0, fma(q1, q1, rr));
            xr = fma(c0, q0, fma(c1, q1, xr));  // (q = 0 outside the mesh)
            sx += (a0 ? c0 : 0.0) + (a1 ? c1 : 0.0);
        }
        rr = warp_sum(rr);
        sx = warp_sum(sx);
        xr = warp_sum(xr);
        if (lane == 0) { part[buf][0][warp] = rr; part[buf][1][warp] = sx; part[buf][2][warp] = xr; }
    }
    __syncthreads();
    if (nb > 0) flush(b0 + nb - 1, (nb - 1) & 1);
}

// Terminal-source solves deliver ONE number, Z[s,s] = b^T L^+ b, and stop early because the CG error of b^T x_k is the
// SQUARE of the energy-norm error -- but only when x_0 = 0: from a guess, b^T (x - x_k) = e_k^T L x_0 + e_k^T L e_k is
// first order again.  The energy form of the same number, E(x_k) = 2 b^T x_k - x_k^T L x_k, is second order from any
// starting point, and CG climbs it by exactly alpha_j rho_j per iteration (Hestenes & Stiefel: ||x - x_j||_L^2 -
// ||x - x_{j+1}||_L^2 = alpha_j rho_j, rho_j = r_j . z_j), so
//     Z[s,s] ~ E(x_k) = E(x_0) + sum_{j<k} alpha_j rho_j,    E(x_0) = b^T x_0 + x_0^T r_0,
// with b^T x_0 = x_0[s] - mean(x_0): the dot x_0 . r_0 is reduced by k_guess_rhs while both are in registers, the sum by
// k_scal_alpha -- no pass over a vector.  (The round's first version evaluated x_0 . r_k from the last residual: one
// more table evaluation and one more vector read per terminal right-hand side, 3 us each at 1024^2, and the
// expected-last probe had to write r_k for it.)  A right-hand side whose guess was rejected started from x_0 = 0:
// b^T x_k is second order there.
__global__ void k_finish_term_guess(GuessTable tab, int pitch, const int* __restrict__ node, const int* __restrict__ src,
                                    const int* __restrict__ keep, const double* __restrict__ sumx, const double* __restrict__ xr0,
                                    const double* __restrict__ arho, double inv_n2, const double* __restrict__ xown,
                                    const double* __restrict__ xmean, int ntsv, double* __restrict__ zdiag, int B) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    double z = xown[b] - xmean[b];
    if (keep[b]) {
        const int so = node[src[b]], ys = so / pitch, xs = so % pitch;
        z = (guess_x0(tab, ys, xs, ys, xs) - sumx[b] * inv_n2) + xr0[b] + arho[b];
    }
    zdiag[src[b] - ntsv] = z;
}

// keep[b] = 1 if the guess of right-hand side b is used (it at least halves the residual), else 0;
// rrk[b] = ||r0||^2 of the starting point the right-hand side ends up with
__global__ void k_guess_check(const double* __restrict__ rr0, double bnorm2, int* __restrict__ keep, double* __restrict__ rrk, int B) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const bool use = rr0[b] <= 0.25 * bnorm2;
    keep[b] = use ? 1 : 0;
    rrk[b] = use ? rr0[b] : bnorm2;
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
