// S1, second-generation stencil kernels: register-resident overlapped tiles.
//
// A 256-thread block owns an extended tile of EW x EH = 32 x 64 nodes (interior (32-2H) x (64-2H),
// halo H recomputed redundantly).  Warp w owns rows 8w..8w+7 of the tile and lane l owns column l:
// every thread keeps, for its 8 nodes, the iterate z, the right-hand side r and the stencil
// coefficients in REGISTERS for the whole kernel; the coefficients are loaded once and reused for
// the G right-hand sides the block loops over.  Left / right neighbours come from the adjacent
// lanes by warp shuffles (a warp spans the full tile width, so no lane ever needs another warp in
// x); only the first and last row of each strip go through a double-buffered shared-memory
// exchange (2 stores + 2 loads and one __syncthreads per sweep).
//
// Smoother: nu steps of Richardson iteration on D^-1 L with the reciprocals of the Chebyshev nodes
// of [2/ratio, 2] as step lengths -- the same polynomial as nu Chebyshev semi-iteration steps, but
// with no direction vector to carry:   z <- (1 - w_k) z + w_k D^-1 (r + sum_nb g_nb z_nb).
#pragma once
#include "common.cuh"

namespace pdn {

#ifndef PDN_T2_R
#define PDN_T2_R 4
#endif
#ifndef PDN_T2_WARPS
#define PDN_T2_WARPS 16
#endif
#ifndef PDN_T2_MINB
#define PDN_T2_MINB 1
#endif
constexpr int T2_R = PDN_T2_R, T2_WARPS = PDN_T2_WARPS, T2_MINB = PDN_T2_MINB;
constexpr int T2_EW = 32, T2_EH = T2_R * T2_WARPS, T2_THREADS = 32 * T2_WARPS;
constexpr unsigned FULL = 0xffffffffu;

struct ChebR {
    int nu;
    double w[MAX_NU];  // step lengths 1 / lambda_k
};

struct Strip {  // per-thread geometry and coefficients
    int lane, warp, gx, gy0;
    unsigned in;  // bit i: node i of the strip lies inside the mesh
    double gE[T2_R], gW[T2_R], gS[T2_R], gN0, dinv[T2_R];
};

// cp.async (LDGSTS) staging: every thread prefetches ITS OWN 8 nodes of the next right-hand side into
// its own shared-memory slots while the block computes the current one; no barrier is needed to
// consume them (a thread only ever reads the slots it filled), and no registers are tied up.
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(sa), "l"(gsrc));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// slot of (stage, array a of NARR, strip node i) for this thread; consecutive threads -> consecutive words
template <int NARR>
__device__ __forceinline__ double* slot(double* stage_mem, int stage, int a, int i) {
    return stage_mem + ((size_t)((stage * NARR + a) * T2_R + i)) * T2_THREADS + threadIdx.x;
}

struct Exch {  // shared-memory exchange of strip boundary rows, double buffered
    double top[2][T2_WARPS][32];
    double bot[2][T2_WARPS][32];
};

template <bool NEED_DINV>
__device__ __forceinline__ void strip_init(Strip& s, const Level& L, int x0, int y0) {
    s.lane = threadIdx.x & 31;
    s.warp = threadIdx.x >> 5;
    s.gx = x0 + s.lane;
    s.gy0 = y0 + T2_R * s.warp;
    const bool xin = s.gx >= 0 && s.gx < L.nx;
    s.in = 0;
#pragma unroll
    for (int i = 0; i < T2_R; ++i) {
        const int gy = s.gy0 + i;
        const bool in = xin && gy >= 0 && gy < L.ny;
        if (in) s.in |= 1u << i;
        const size_t gi = (size_t)gy * L.nx + s.gx;
        s.gE[i] = in ? __ldg(L.gx + gi) : 0.0;
        s.gS[i] = in ? __ldg(L.gy + gi) : 0.0;
        s.gW[i] = (in && s.gx > 0) ? __ldg(L.gx + gi - 1) : 0.0;
        s.dinv[i] = (in && NEED_DINV) ? __ldg(L.dinv + gi) : 0.0;
    }
    const int gyn = s.gy0 - 1;
    s.gN0 = (xin && gyn >= 0 && gyn < L.ny) ? __ldg(L.gy + (size_t)gyn * L.nx + s.gx) : 0.0;
}

// t[i] = sum over the four neighbours of g_nb * z_nb.  One barrier; `cur` flips.
__device__ __forceinline__ void neighbour_sum(Exch& x, int& cur, const Strip& s, const double (&z)[T2_R],
                                              double (&t)[T2_R]) {
    x.top[cur][s.warp][s.lane] = z[0];
    x.bot[cur][s.warp][s.lane] = z[T2_R - 1];
    __syncthreads();
    const double zt = s.warp > 0 ? x.bot[cur][s.warp - 1][s.lane] : 0.0;
    const double zb = s.warp < T2_WARPS - 1 ? x.top[cur][s.warp + 1][s.lane] : 0.0;
    cur ^= 1;
#pragma unroll
    for (int i = 0; i < T2_R; ++i) {
        const double zl = __shfl_up_sync(FULL, z[i], 1);
        const double zr = __shfl_down_sync(FULL, z[i], 1);
        const double zu = i == 0 ? zt : z[i - 1];
        const double zd = i == T2_R - 1 ? zb : z[i + 1];
        const double gN = i == 0 ? s.gN0 : s.gS[i - 1];
        double a = s.gE[i] * zr;
        a = fma(s.gW[i], zl, a);
        a = fma(s.gS[i], zd, a);
        a = fma(gN, zu, a);
        t[i] = a;
    }
}

// r is read from the thread's own staging slots (rs[i * T2_THREADS]) to keep it out of the register file
__device__ __forceinline__ void smooth_step(Exch& x, int& cur, const Strip& s, const double* rs, double (&z)[T2_R],
                                            double w) {
    double t[T2_R];
    neighbour_sum(x, cur, s, z, t);
    const double a = 1.0 - w;
#pragma unroll
    for (int i = 0; i < T2_R; ++i) z[i] = fma(w * s.dinv[i], rs[i * T2_THREADS] + t[i], a * z[i]);
}

// ---------------------------------------------------------------------------------------------
// Down stage (mathematics as k_down in stencil.cuh):
//   [r = r_in - alpha q ; rr += r.r]   z = S_nu(0, r)   rc = R (r - L z)
// grid = (tiles_x, tiles_y, ceil(B / G)); the block loops over G right-hand sides.
template <int NU, bool FUSED>
__global__ void __launch_bounds__(T2_THREADS, T2_MINB)
k_down2(Level L, ChebR ch, const double* __restrict__ r_in, const double* __restrict__ q,
        const double* __restrict__ alpha, double* __restrict__ r_out, double* __restrict__ z_out,
        double* __restrict__ rc, int cny, int cnx, double* __restrict__ rr_acc, int B, int G) {
    constexpr int H = NU, IW = T2_EW - 2 * H, IH = T2_EH - 2 * H, PAR = H & 1;
    __shared__ Exch x;
    __shared__ double red[32];
    const int x0 = blockIdx.x * IW - H, y0 = blockIdx.y * IH - H;
    Strip s;
    strip_init<true>(s, L, x0, y0);
    const size_t plane = (size_t)L.ny * L.nx, cplane = (size_t)cny * cnx;
    const bool xint = s.lane >= H && s.lane < H + IW;
    const int ey0 = T2_R * s.warp;
    unsigned interior = 0;  // bit i: node i is an interior node of the tile and inside the mesh
#pragma unroll
    for (int i = 0; i < T2_R; ++i)
        if (xint && ey0 + i >= H && ey0 + i < H + IH && ((s.in >> i) & 1)) interior |= 1u << i;
    const size_t goff = (size_t)s.gy0 * L.nx + s.gx;
    const int b_end = min(B, (int)(blockIdx.z + 1) * G);
    constexpr int NARR = FUSED ? 2 : 1;
    extern __shared__ double stage_mem[];
#pragma unroll
    for (int st = 0; st < 2; ++st)
#pragma unroll
        for (int a = 0; a < NARR; ++a)
#pragma unroll
            for (int i = 0; i < T2_R; ++i)
                if (!((s.in >> i) & 1)) *slot<NARR>(stage_mem, st, a, i) = 0.0;  // nodes outside the mesh stay 0
    auto prefetch = [&](int b, int st) {
#pragma unroll
        for (int i = 0; i < T2_R; ++i)
            if ((s.in >> i) & 1) {
                cp_async8(slot<NARR>(stage_mem, st, 0, i), r_in + b * plane + goff + (size_t)i * L.nx);
                if (FUSED) cp_async8(slot<NARR>(stage_mem, st, 1, i), q + b * plane + goff + (size_t)i * L.nx);
            }
        cp_async_commit();
    };
    int cur = 0, st = 0;
    prefetch(blockIdx.z * G, 0);
    for (int b = blockIdx.z * G; b < b_end; ++b, st ^= 1) {
        if (b + 1 < b_end) {
            prefetch(b + 1, st ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        double* rs = slot<NARR>(stage_mem, st, 0, 0);
        double z[T2_R];
        const double al = FUSED ? alpha[b] : 0.0;
        double rr = 0.0;
#pragma unroll
        for (int i = 0; i < T2_R; ++i) {
            double v = rs[i * T2_THREADS];
            if (FUSED) {
                v = fma(-al, *slot<NARR>(stage_mem, st, 1, i), v);
                rs[i * T2_THREADS] = v;
                if ((interior >> i) & 1) {
                    r_out[b * plane + goff + (size_t)i * L.nx] = v;
                    rr = fma(v, v, rr);
                }
            }
            z[i] = ch.w[0] * s.dinv[i] * v;
        }
#pragma unroll
        for (int k = 1; k < NU; ++k) smooth_step(x, cur, s, rs, z, ch.w[k]);
        double t[T2_R], res[T2_R];
        neighbour_sum(x, cur, s, z, t);
#pragma unroll
        for (int i = 0; i < T2_R; ++i) {
            const double gN = i == 0 ? s.gN0 : s.gS[i - 1];
            const double dg = (s.gE[i] + s.gW[i]) + (s.gS[i] + gN);
            res[i] = fma(-dg, z[i], rs[i * T2_THREADS] + t[i]);
            if ((interior >> i) & 1) z_out[b * plane + goff + (size_t)i * L.nx] = z[i];
        }
        // restriction: sum over 2x2 aggregates.  Global coordinates of strip row 0 / lane 0 have the
        // parity of H, so with H odd the aggregates straddle strips and lanes by one node.
        double below0 = 0.0;
        if (PAR) {
            x.top[cur][s.warp][s.lane] = res[0];
            __syncthreads();
            below0 = s.warp < T2_WARPS - 1 ? x.top[cur][s.warp + 1][s.lane] : 0.0;
            cur ^= 1;
        }
#pragma unroll
        for (int j = 0; j < T2_R / 2; ++j) {
            const int i0 = 2 * j + PAR;  // first fine row of the aggregate inside this strip
            const double lower = (i0 + 1 < T2_R) ? res[(i0 + 1) % T2_R] : below0;
            double v = res[i0] + lower;
            v += __shfl_down_sync(FULL, v, 1);
            const int ey = ey0 + i0, gy = s.gy0 + i0;
            const bool writer = ((s.lane + PAR) & 1) == 0 && s.lane >= H && s.lane + 1 < H + IW && ey >= H &&
                                ey + 1 < H + IH;
            if (writer) {
                const int gcy = gy >> 1, gcx = s.gx >> 1;
                if (gcy < cny && gcx < cnx) rc[b * cplane + (size_t)gcy * cnx + gcx] = v;
            }
        }
        if (FUSED) {
            rr = block_sum(rr, red);
            if (threadIdx.x == 0) atomicAdd(rr_acc + b, rr);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Up stage:  z = z_in + P e_c ;  z = S_nu(z, r) ;  [rz += r.z]
template <int NU, bool DOT>
__global__ void __launch_bounds__(T2_THREADS, T2_MINB)
k_up2(Level L, ChebR ch, const double* __restrict__ r_g, const double* __restrict__ z_in,
      const double* __restrict__ ec, int cny, int cnx, double* __restrict__ z_out, double* __restrict__ rz_acc,
      int B, int G) {
    constexpr int H = NU, IW = T2_EW - 2 * H, IH = T2_EH - 2 * H;
    __shared__ Exch x;
    __shared__ double red[32];
    const int x0 = blockIdx.x * IW - H, y0 = blockIdx.y * IH - H;
    Strip s;
    strip_init<true>(s, L, x0, y0);
    const size_t plane = (size_t)L.ny * L.nx, cplane = (size_t)cny * cnx;
    const bool xint = s.lane >= H && s.lane < H + IW;
    const int ey0 = T2_R * s.warp;
    unsigned interior = 0;
#pragma unroll
    for (int i = 0; i < T2_R; ++i)
        if (xint && ey0 + i >= H && ey0 + i < H + IH && ((s.in >> i) & 1)) interior |= 1u << i;
    const size_t goff = (size_t)s.gy0 * L.nx + s.gx;
    const int b_end = min(B, (int)(blockIdx.z + 1) * G);
    constexpr int NARR = 3;  // r, z_in, coarse correction
    extern __shared__ double stage_mem[];
#pragma unroll
    for (int st = 0; st < 2; ++st)
#pragma unroll
        for (int a = 0; a < NARR; ++a)
#pragma unroll
            for (int i = 0; i < T2_R; ++i)
                if (!((s.in >> i) & 1)) *slot<NARR>(stage_mem, st, a, i) = 0.0;
    auto prefetch = [&](int b, int st) {
#pragma unroll
        for (int i = 0; i < T2_R; ++i)
            if ((s.in >> i) & 1) {
                cp_async8(slot<NARR>(stage_mem, st, 0, i), r_g + b * plane + goff + (size_t)i * L.nx);
                cp_async8(slot<NARR>(stage_mem, st, 1, i), z_in + b * plane + goff + (size_t)i * L.nx);
                cp_async8(slot<NARR>(stage_mem, st, 2, i),
                          ec + b * cplane + (size_t)((s.gy0 + i) >> 1) * cnx + (s.gx >> 1));
            }
        cp_async_commit();
    };
    int cur = 0, st = 0;
    prefetch(blockIdx.z * G, 0);
    for (int b = blockIdx.z * G; b < b_end; ++b, st ^= 1) {
        if (b + 1 < b_end) {
            prefetch(b + 1, st ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        const double* rs = slot<NARR>(stage_mem, st, 0, 0);
        double z[T2_R];
#pragma unroll
        for (int i = 0; i < T2_R; ++i) z[i] = *slot<NARR>(stage_mem, st, 1, i) + *slot<NARR>(stage_mem, st, 2, i);
#pragma unroll
        for (int k = 0; k < NU; ++k) smooth_step(x, cur, s, rs, z, ch.w[NU - 1 - k]);
        double rz = 0.0;
#pragma unroll
        for (int i = 0; i < T2_R; ++i) {
            if ((interior >> i) & 1) {
                z_out[b * plane + goff + (size_t)i * L.nx] = z[i];
                rz = fma(rs[i * T2_THREADS], z[i], rz);
            }
        }
        if (DOT) {
            rz = block_sum(rz, red);
            if (threadIdx.x == 0) atomicAdd(rz_acc + b, rz);
        }
    }
}

}  // namespace pdn
