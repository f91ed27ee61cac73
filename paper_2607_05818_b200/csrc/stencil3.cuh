// S1: batched matrix-free multigrid-PCG kernels on the per-tier 2D 5-point stencil (sm_100a).
//
// Layout.  Every vector is a batch of pitched planes v[b][y][pitch] (b = right-hand side).
//
// Tiling.  A block of W warps owns an extended tile of 64 x (R*W) nodes: interior
// (64-2H) x (R*W-2H) plus a halo of H nodes that is recomputed redundantly, so a whole multigrid
// stage (all its sweeps) runs on chip with no exchange between blocks.  Lane l of warp w owns the
// 2 x R patch of columns 2l, 2l+1 and rows R*w .. R*w+R-1:
//   * the iterate and the stencil coefficients of the patch live in REGISTERS for the whole kernel;
//     the coefficients are loaded once per block and reused for the G right-hand sides it loops over;
//   * left / right neighbours come from the adjacent lanes by warp shuffles, the rows above / below
//     the patch through a double-buffered shared-memory exchange with a split-phase mbarrier
//     (publish + arrive, update the rows that need no other warp, wait, update the boundary rows);
//   * the tile + halo of every input vector is fetched by TMA (cp.async.bulk.tensor, 3D box
//     64 x R*W x 1 of a (x, y, rhs) tensor map) into shared memory, two stages, completion on an
//     mbarrier, the fetch of right-hand side j+2 overlapping the sweeps of j and j+1.  Out-of-mesh
//     elements arrive as zeros, and the coefficients there are zero: no boundary cases in the sweeps;
//   * converged right-hand sides are skipped (ActiveList);
//   * global stores are 16-byte (both columns of a patch row), interior only.
//
// Arithmetic.  The V-cycle sweeps act on the symmetrically scaled system (common.cuh: Level):
//   y <- (1-w) y + w (r^ + sum_nb h_nb y_nb),   r^ = s r,   z = s y,
// with r^ and y of the patch in registers; k_pq3 (the CG operator apply) uses the raw conductances.
//
// What bounds these kernels (ncu, profiles/): the shared-memory data pipe (128 B/clk/SM), which TMA
// fills, LDS/STS and the warp shuffles all share -- so every input value crosses it exactly twice
// (TMA write, one LDS), nothing is re-read per sweep, and the per-sweep traffic is the patch perimeter.
#pragma once
#include "common.cuh"

namespace pdn {

constexpr unsigned FULL = 0xffffffffu;
constexpr int T3_EW = 64;
// The coarse correction of a tile is 32 coarse columns starting at x0/2, which may be odd; TMA wants the
// innermost box coordinate 16-byte aligned, so the box starts at the even column below and is 34 wide.
constexpr int T3_ECW = 34;


// T = the type the sweeps compute in: double everywhere by default; float for the V-cycle stages of a context
// created with PDN_PRECOND_F32 (the preconditioner only: the CG operator, residuals and solutions stay FP64).
template <class T> struct Vec2;
template <> struct Vec2<double> { using type = double2; };
template <> struct Vec2<float> { using type = float2; };
template <class T> __device__ __forceinline__ typename Vec2<T>::type mk2(T a, T b);
template <> __device__ __forceinline__ double2 mk2<double>(double a, double b) { return make_double2(a, b); }
template <> __device__ __forceinline__ float2 mk2<float>(float a, float b) { return make_float2(a, b); }

template <int R, class T = double>
struct Patch {  // scaled coefficients of a 2 x R patch
    T hE0[R], hE1[R];  // east of column 0 (= west of column 1), east of column 1
    T hW0[R];          // west of column 0
    T hS0[R], hS1[R];  // south of row i (= north of row i+1)
    T hN0, hN1;        // north of row 0
};

template <int W, class T = double>
struct Exch {  // rows above / below every warp's patch, double buffered; slot 0 of bot and slot W of top stay 0
    typename Vec2<T>::type top[2][W + 1][32];
    typename Vec2<T>::type bot[2][W + 1][32];
};

__device__ __forceinline__ double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void st2(double* p, double2 v) { *reinterpret_cast<double2*>(p) = v; }
__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }

template <int R, int W, class T>
__device__ __forceinline__ void exch_clear(Exch<W, T>& x) {
    for (int i = threadIdx.x; i < 2 * 32; i += 32 * W) {
        x.top[i >> 5][W][i & 31] = mk2<T>(T(0), T(0));
        x.bot[i >> 5][0][i & 31] = mk2<T>(T(0), T(0));
    }
}

// Coefficients of this thread's patch (zeros outside the mesh) and its slots of the scaling tile: two float2
// planes, s_slot[row*32] = s of columns 0, 1 and s_slot[SD_OFF + row*32] = sd of columns 0, 1, so that a stage
// that needs only one of the two reads 8 bytes per lane, not 16.
template <int R, class T>
__device__ __forceinline__ void patch_init(Patch<R, T>& c, const double* __restrict__ pE, const double* __restrict__ pS,
                                           const float2* __restrict__ psc, const Level& L, int gx, int gy0,
                                           float2* s_slot, int sd_off) {
    const bool xin = gx >= 0 && gx < L.pitch;  // gx is even, pitch is even: both columns are addressable
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const int gy = gy0 + i;
        const bool in = xin && gy >= 0 && gy < L.ny;
        const size_t gi = (size_t)gy * L.pitch + gx;
        const double2 z2 = make_double2(0.0, 0.0);
        const double2 e = in ? ldg2(pE + gi) : z2;
        const double2 s = in ? ldg2(pS + gi) : z2;
        c.hE0[i] = (T)e.x; c.hE1[i] = (T)e.y;
        c.hS0[i] = (T)s.x; c.hS1[i] = (T)s.y;
        c.hW0[i] = (T)((in && gx > 0) ? __ldg(pE + gi - 1) : 0.0);
        if (psc) {
            const float4 v = in ? __ldg(reinterpret_cast<const float4*>(psc + gi)) : make_float4(0.f, 0.f, 0.f, 0.f);
            s_slot[i * 32] = make_float2(v.x, v.z);
            s_slot[sd_off + i * 32] = make_float2(v.y, v.w);
        }
    }
    const int gyn = gy0 - 1;
    const double2 nn = (xin && gyn >= 0 && gyn < L.ny) ? ldg2(pS + (size_t)gyn * L.pitch + gx) : make_double2(0.0, 0.0);
    c.hN0 = (T)nn.x; c.hN1 = (T)nn.y;
}

// Split-phase exchange of patch boundary rows between the warps of a block.  `publish` stores the
// patch's first and last row and ARRIVES on an mbarrier; the rows that need nothing from other warps
// are computed next; `collect` waits for everybody's arrival and fetches the rows just above / below.
// Buffers alternate between sweeps, the mbarrier phase flips once per sweep.
template <int W, class T = double>
struct Xchg {
    using T2 = typename Vec2<T>::type;
    Exch<W, T>* x;
    uint64_t* bar;
    int cur;        // buffer of the current sweep
    uint32_t phase; // parity the next collect waits for
    int warp, lane;
    __device__ __forceinline__ void publish(T a0, T a1, T b0, T b1) {
        x->top[cur][warp][lane] = mk2<T>(a0, a1);
        x->bot[cur][warp + 1][lane] = mk2<T>(b0, b1);
        mbar_arrive(bar);
    }
    __device__ __forceinline__ void collect(T2& up, T2& dn) {
        mbar_wait(bar, phase);
        up = x->bot[cur][warp][lane];
        dn = x->top[cur][warp + 1][lane];
        cur ^= 1;
        phase ^= 1;
    }
};

// t = add + sum over the four neighbours of h_nb * y_nb for row i of the patch, whose own values are
// (c0, c1), with the rows above (u0, u1) and below (d0, d1) given explicitly.
template <int R, class T>
__device__ __forceinline__ void row_sum(const Patch<R, T>& c, int i, T c0, T c1, T u0, T u1,
                                        T d0, T d1, T add0, T add1, T& t0, T& t1) {
    const T yl = __shfl_up_sync(FULL, c1, 1);    // right column of the lane to the left
    const T yr = __shfl_down_sync(FULL, c0, 1);  // left column of the lane to the right
    const T n0 = i == 0 ? c.hN0 : c.hS0[i == 0 ? 0 : i - 1], n1 = i == 0 ? c.hN1 : c.hS1[i == 0 ? 0 : i - 1];
    T a = fma(c.hE0[i], c1, add0);
    a = fma(c.hW0[i], yl, a);
    a = fma(c.hS0[i], d0, a);
    t0 = fma(n0, u0, a);
    T b = fma(c.hE1[i], yr, add1);
    b = fma(c.hE0[i], c0, b);
    b = fma(c.hS1[i], d1, b);
    t1 = fma(n1, u1, b);
}

// One Richardson step  y <- (1-w) y + w (r^ + N y)  on the patch, in place.  Rows 1..R-2 need only this
// thread's (and, by shuffle, this warp's) values: they are updated between publish and collect, top to
// bottom, the old value of the row above carried in registers; rows 0 and R-1 follow the collect.
template <int R, int W, class T>
__device__ __forceinline__ void smooth_step(Xchg<W, T>& xc, const Patch<R, T>& c, T (&y0)[R], T (&y1)[R],
                                            const T (&rh0)[R], const T (&rh1)[R], T w) {
    static_assert(R >= 2, "patch needs two rows");
    xc.publish(y0[0], y1[0], y0[R - 1], y1[R - 1]);
    const T a = T(1) - w;
    const T f0 = y0[0], f1 = y1[0];          // old first row
    const T s0 = y0[R > 2 ? 1 : 0], s1 = y1[R > 2 ? 1 : 0];  // old second row (below neighbour of row 0)
    const T l0 = y0[R - 1], l1 = y1[R - 1];  // old last row
    T pu0 = f0, pu1 = f1;
#pragma unroll
    for (int i = 1; i < R - 1; ++i) {
        T t0, t1;
        row_sum<R, T>(c, i, y0[i], y1[i], pu0, pu1, y0[i + 1], y1[i + 1], rh0[i], rh1[i], t0, t1);
        pu0 = y0[i]; pu1 = y1[i];
        y0[i] = fma(w, t0, a * y0[i]);
        y1[i] = fma(w, t1, a * y1[i]);
    }
    // pu = old row R-2 (or the old first row if R == 2)
    typename Vec2<T>::type up, dn;
    xc.collect(up, dn);
    T t0, t1, v0, v1;
    row_sum<R, T>(c, 0, f0, f1, up.x, up.y, R > 2 ? s0 : l0, R > 2 ? s1 : l1, rh0[0], rh1[0], t0, t1);
    row_sum<R, T>(c, R - 1, l0, l1, pu0, pu1, dn.x, dn.y, rh0[R - 1], rh1[R - 1], v0, v1);
    y0[0] = fma(w, t0, a * f0);
    y1[0] = fma(w, t1, a * f1);
    y0[R - 1] = fma(w, v0, a * l0);
    y1[R - 1] = fma(w, v1, a * l1);
}

// t = add + N y for every row of the patch (y unchanged): the residual / operator-apply variant.
// `hook` runs right after this warp has published its boundary rows (work that needs no other warp).
struct NoHook { __device__ __forceinline__ void operator()() const {} };
template <int R, int W, class T, class F = NoHook>
__device__ __forceinline__ void apply_step(Xchg<W, T>& xc, const Patch<R, T>& c, const T (&y0)[R], const T (&y1)[R],
                                           const T (&a0)[R], const T (&a1)[R], T (&t0)[R],
                                           T (&t1)[R], F&& hook = F()) {
    xc.publish(y0[0], y1[0], y0[R - 1], y1[R - 1]);
    hook();
#pragma unroll
    for (int i = 1; i < R - 1; ++i)
        row_sum<R, T>(c, i, y0[i], y1[i], y0[i - 1], y1[i - 1], y0[i + 1], y1[i + 1], a0[i], a1[i], t0[i], t1[i]);
    typename Vec2<T>::type up, dn;
    xc.collect(up, dn);
    row_sum<R, T>(c, 0, y0[0], y1[0], up.x, up.y, y0[1], y1[1], a0[0], a1[0], t0[0], t1[0]);
    row_sum<R, T>(c, R - 1, y0[R - 1], y1[R - 1], y0[R - 2], y1[R - 2], dn.x, dn.y, a0[R - 1], a1[R - 1], t0[R - 1], t1[R - 1]);
}

template <int R, int W, int H>
struct Geom {
    static constexpr int EH = R * W, IW = T3_EW - 2 * H, IH = EH - 2 * H, TILE = EH * T3_EW, THREADS = 32 * W;
    static constexpr int ETILE = ((EH / 2) * T3_ECW + 15) & ~15;  // coarse-correction tile of the up stage (128-byte multiple)
    static constexpr uint32_t TILE_BYTES = TILE * sizeof(double), ETILE_BYTES = ETILE * sizeof(double);
    static constexpr uint32_t EBOX_BYTES = (EH / 2) * T3_ECW * sizeof(double);  // what the TMA box delivers
    static_assert(R % 2 == 0 && H % 2 == 0, "2x2 aggregates must not straddle patches");
    static_assert(IW > 0 && IH > 0, "halo too deep for the tile");
};

// The right-hand sides of [b0, b0 + nmax) that are still iterating (all of them if active == nullptr), in
// order, for every thread of the block.  Converged right-hand sides are frozen: no kernel touches their
// vectors again.  Call before the block's first __syncthreads.
constexpr int T3_MAX_G = 64;     // V-cycle stages: a block's set-up (coefficients, scaling tile) is spread over up to 64
constexpr int T3_MAX_G_PQ = 32;  // operator apply: lighter set-up; measured 2 % slower with 64

struct ActiveList {
    int b[T3_MAX_G];
    double s[T3_MAX_G];  // the per-right-hand-side scalar of the kernel (alpha / beta), staged once per block so that
    int n;               // the loop over right-hand sides has no dependent global load in front of its first FMA
};
__device__ __forceinline__ void active_list_build(ActiveList& al, const int* __restrict__ active, int b0, int nmax,
                                                  const double* __restrict__ scal = nullptr) {
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        int cnt = 0;
        for (int base = 0; base < nmax; base += 32) {
            const int j = base + lane;
            const bool a = j < nmax && (active == nullptr || active[b0 + j] != 0);
            const unsigned m = __ballot_sync(FULL, a);
            if (a) {
                const int slot = cnt + __popc(m & ((1u << lane) - 1u));
                al.b[slot] = b0 + j;
                al.s[slot] = scal ? scal[b0 + j] : 0.0;
            }
            cnt += __popc(m);
        }
        if (lane == 0) al.n = cnt;
    }
}

__host__ __device__ constexpr int halo_of(int nu) { return (nu + 1) & ~1; }

// bit i: row i of the patch is an interior row of the tile and inside the mesh (columns too)
template <int R, int H, int IW, int IH>
__device__ __forceinline__ unsigned interior_mask(const Level& L, int lane, int warp, int gx, int gy0) {
    const bool xint = 2 * lane >= H && 2 * lane < H + IW && gx < L.nx;
    unsigned m = 0;
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const int ey = R * warp + i;
        if (xint && ey >= H && ey < H + IH && gy0 + i < L.ny) m |= 1u << i;
    }
    return m;
}

// ---------------------------------------------------------------------------------------------
// Down stage of the V-cycle on one level (fused with the CG residual update on level 0):
//   [r = r_in - alpha q ; rr += r.r]   y = S_nu(0, r^)   rc = R sd (r^ - A^ y)
// y (the scaled iterate) is written to y_out for the up stage; R sums 2x2 aggregates.
// grid = (tiles_x, tiles_y, ceil(B / G)); the block loops over G right-hand sides, two TMA stages.
template <int R, int W, int NU, bool FUSED, class T = double>
__global__ void __launch_bounds__(32 * W, 1)
k_down3(const __grid_constant__ CUtensorMap tm_r, const __grid_constant__ CUtensorMap tm_q, Level L, ChebR ch,
        const double* __restrict__ alpha, double* __restrict__ r_out, double* __restrict__ y_out,
        double* __restrict__ rc, int cny, int cnx, int cpitch, double* __restrict__ rr_acc, int B, int G, const int* __restrict__ active) {
    constexpr int H = halo_of(NU);
    using Gm = Geom<R, W, H>;
    extern __shared__ __align__(128) double smem_dyn[];
    double* rbuf = smem_dyn;                                   // 2 stages
    double* qbuf = rbuf + 2 * Gm::TILE;                        // 2 stages (FUSED only)
    float2* sc = reinterpret_cast<float2*>(qbuf + (FUSED ? 2 * Gm::TILE : 0));
    constexpr int SD_OFF = Gm::EH * 32;
    Exch<W, T>& x = *reinterpret_cast<Exch<W, T>*>(sc + 2 * SD_OFF);
    __shared__ uint64_t mbar[3];  // two TMA stages + the row-exchange barrier

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int x0 = blockIdx.x * Gm::IW - H, y0 = blockIdx.y * Gm::IH - H;
    const int gx = x0 + 2 * lane, gy0 = y0 + R * warp;
    const int slot0 = (R * warp) * T3_EW + 2 * lane;
    float2* sc_slot = sc + (R * warp) * 32 + lane;
    Patch<R, T> c;
    patch_init<R, T>(c, L.hE, L.hS, L.sc, L, gx, gy0, sc_slot, SD_OFF);
    exch_clear<R, W, T>(x);
    const unsigned interior = interior_mask<R, H, Gm::IW, Gm::IH>(L, lane, warp, gx, gy0);
    const size_t plane = (size_t)L.ny * L.pitch, cplane = (size_t)cny * cpitch;
    const size_t goff = (size_t)gy0 * L.pitch + gx;
    const ptrdiff_t coff = (ptrdiff_t)(gy0 >> 1) * cpitch + (gx >> 1);  // coarse node of the patch's first 2x2 aggregate (gy0, gx even)
    __shared__ ActiveList al;
    active_list_build(al, active, blockIdx.z * G, min(G, B - (int)blockIdx.z * G), FUSED ? alpha : nullptr);
    if (threadIdx.x == 0) {
        mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); mbar_init(&mbar[2], 32 * W);
        mbar_fence_init();
    }
    __syncthreads();
    const int nb = al.n;
    auto fetch = [&](int j) {  // thread 0 only
        const int st = j & 1;
        mbar_expect_tx(&mbar[st], (FUSED ? 2 : 1) * Gm::TILE_BYTES);
        tma_load_3d(rbuf + st * Gm::TILE, &tm_r, x0, y0, al.b[j], &mbar[st]);
        if (FUSED) tma_load_3d(qbuf + st * Gm::TILE, &tm_q, x0, y0, al.b[j], &mbar[st]);
    };
    if (threadIdx.x == 0 && nb > 0) {  // nb == 0: every right-hand side of the group has converged
        fetch(0);
        if (nb > 1) fetch(1);
    }
    Xchg<W, T> xc{&x, &mbar[2], 0, 0u, warp, lane};
    for (int j = 0; j < nb; ++j) {
        const int b = al.b[j], st = j & 1;
        mbar_wait(&mbar[st], (j >> 1) & 1);
        const double alj = FUSED ? al.s[j] : 0.0;
        T y0r[R], y1r[R], rh0[R], rh1[R];
        double rr = 0.0;
        double* rp = FUSED ? r_out + b * plane + goff : nullptr;
#pragma unroll
        for (int i = 0; i < R; ++i) {
            double2 r = ld2(rbuf + st * Gm::TILE + slot0 + i * T3_EW);
            if (FUSED) {
                const double2 q = ld2(qbuf + st * Gm::TILE + slot0 + i * T3_EW);
                r.x = fma(-alj, q.x, r.x);
                r.y = fma(-alj, q.y, r.y);
                if ((interior >> i) & 1) {
                    st2(rp, r);
                    rr = fma(r.x, r.x, rr);
                    rr = fma(r.y, r.y, rr);
                }
                rp += L.pitch;
            }
            const float2 s2 = sc_slot[i * 32];
            rh0[i] = (T)s2.x * (T)r.x;
            rh1[i] = (T)s2.y * (T)r.y;
            y0r[i] = (T)ch.w[0] * rh0[i];
            y1r[i] = (T)ch.w[0] * rh1[i];
        }
        if (FUSED) {  // ||r||^2: the shuffle chain overlaps the sweeps that follow
            rr = warp_sum(rr);
            if (lane == 0) atomicAdd(rr_acc + b, rr);
        }
        // once thread 0 is past the first row exchange of this iteration every thread has arrived there,
        // i.e. has consumed the stage: thread 0 may refill it with right-hand side j+2
#pragma unroll
        for (int k = 1; k < NU; ++k) {
            smooth_step<R, W, T>(xc, c, y0r, y1r, rh0, rh1, (T)ch.w[k]);
            if (k == 1 && threadIdx.x == 0 && j + 2 < nb) fetch(j + 2);
        }
        T t0[R], t1[R];
        // y is final: its stores leave right after this warp has published its boundary rows and drain (an SM stores
        // 32 B/clk: measured) while the residual is computed, instead of in one burst with rc at the end
        apply_step<R, W, T>(xc, c, y0r, y1r, rh0, rh1, t0, t1, [&] {
            double* yp = y_out + b * plane + goff;
#pragma unroll
            for (int i = 0; i < R; ++i) {
                if ((interior >> i) & 1) st2(yp, make_double2((double)y0r[i], (double)y1r[i]));
                yp += L.pitch;
            }
        });
        if (NU == 1 && threadIdx.x == 0 && j + 2 < nb) fetch(j + 2);
        // residual of the unscaled system at the patch nodes, summed over 2x2 aggregates
        double* rcp = rc + b * cplane + coff;
#pragma unroll
        for (int i = 0; i < R; i += 2) {
            const float2 sa = sc_slot[SD_OFF + i * 32], sb = sc_slot[SD_OFF + (i + 1) * 32];
            T v = (T)sa.x * (t0[i] - y0r[i]);
            v = fma((T)sa.y, t1[i] - y1r[i], v);
            v = fma((T)sb.x, t0[i + 1] - y0r[i + 1], v);
            v = fma((T)sb.y, t1[i + 1] - y1r[i + 1], v);
            if ((interior >> i) & 1) *rcp = (double)v;  // rows i and i+1 are interior together (H, R, y0 even)
            rcp += cpitch;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Up stage:  y = y_in + sd P e_c ;  y = S_nu(y, r^) ;  z = s y ;  [rz += r.z]
// P = piecewise-constant prolongation (fine (y,x) takes coarse (y/2, x/2)).
template <int R, int W, int NU, bool DOT, class T = double>
__global__ void __launch_bounds__(32 * W, 1)
k_up3(const __grid_constant__ CUtensorMap tm_r, const __grid_constant__ CUtensorMap tm_y,
      const __grid_constant__ CUtensorMap tm_e, Level L, ChebR ch, double* __restrict__ z_out,
      double* __restrict__ rz_acc, int B, int G, const int* __restrict__ active) {
    constexpr int H = halo_of(NU);
    using Gm = Geom<R, W, H>;
    extern __shared__ __align__(128) double smem_dyn[];
    double* rbuf = smem_dyn;             // 2 stages each
    double* ybuf = rbuf + 2 * Gm::TILE;
    double* ebuf = ybuf + 2 * Gm::TILE;  // T3_ECW x EH/2 per stage
    float2* sc = reinterpret_cast<float2*>(ebuf + 2 * Gm::ETILE);
    constexpr int SD_OFF = Gm::EH * 32;
    Exch<W, T>& x = *reinterpret_cast<Exch<W, T>*>(sc + 2 * SD_OFF);
    __shared__ uint64_t mbar[3];  // two TMA stages + the row-exchange barrier

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int x0 = blockIdx.x * Gm::IW - H, y0 = blockIdx.y * Gm::IH - H;
    const int gx = x0 + 2 * lane, gy0 = y0 + R * warp;
    const int slot0 = (R * warp) * T3_EW + 2 * lane;
    float2* sc_slot = sc + (R * warp) * 32 + lane;
    Patch<R, T> c;
    patch_init<R, T>(c, L.hE, L.hS, L.sc, L, gx, gy0, sc_slot, SD_OFF);
    exch_clear<R, W, T>(x);
    const unsigned interior = interior_mask<R, H, Gm::IW, Gm::IH>(L, lane, warp, gx, gy0);
    const size_t plane = (size_t)L.ny * L.pitch;
    const size_t goff = (size_t)gy0 * L.pitch + gx;
    __shared__ ActiveList al;
    active_list_build(al, active, blockIdx.z * G, min(G, B - (int)blockIdx.z * G));
    const int cx0 = (x0 >> 1) & ~1;                 // even coarse column at or below x0/2 (x0 is even)
    const int eslot = (x0 >> 1) - cx0 + lane;       // this lane's coarse column inside the box
    if (threadIdx.x == 0) {
        mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); mbar_init(&mbar[2], 32 * W);
        mbar_fence_init();
    }
    __syncthreads();
    const int nb = al.n;
    auto fetch = [&](int j) {  // thread 0 only
        const int st = j & 1;
        mbar_expect_tx(&mbar[st], 2 * Gm::TILE_BYTES + Gm::EBOX_BYTES);
        tma_load_3d(rbuf + st * Gm::TILE, &tm_r, x0, y0, al.b[j], &mbar[st]);
        tma_load_3d(ybuf + st * Gm::TILE, &tm_y, x0, y0, al.b[j], &mbar[st]);
        tma_load_3d(ebuf + st * Gm::ETILE, &tm_e, cx0, y0 / 2, al.b[j], &mbar[st]);
    };
    if (threadIdx.x == 0 && nb > 0) {  // nb == 0: every right-hand side of the group has converged
        fetch(0);
        if (nb > 1) fetch(1);
    }
    Xchg<W, T> xc{&x, &mbar[2], 0, 0u, warp, lane};
    double rz_pend = 0.0;  // r.z partial of the previous right-hand side: reduced while the next one sweeps
    int b_pend = -1;
    for (int j = 0; j < nb; ++j) {
        const int b = al.b[j], st = j & 1;
        mbar_wait(&mbar[st], (j >> 1) & 1);
        T y0r[R], y1r[R], rh0[R], rh1[R];
        T ec[R / 2];  // one coarse correction per pair of rows (R and H are even: rows 2k, 2k+1 share a coarse row)
#pragma unroll
        for (int k = 0; k < R / 2; ++k) ec[k] = (T)ebuf[st * Gm::ETILE + ((R * warp) / 2 + k) * T3_ECW + eslot];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 r = ld2(rbuf + st * Gm::TILE + slot0 + i * T3_EW);
            const double2 yin = ld2(ybuf + st * Gm::TILE + slot0 + i * T3_EW);
            const T e = ec[i >> 1];
            const float2 s2 = sc_slot[i * 32], d2 = sc_slot[SD_OFF + i * 32];
            rh0[i] = (T)s2.x * (T)r.x;
            rh1[i] = (T)s2.y * (T)r.y;
            y0r[i] = fma((T)d2.x, e, (T)yin.x);
            y1r[i] = fma((T)d2.y, e, (T)yin.y);
        }
        if (DOT && b_pend >= 0) {
            rz_pend = warp_sum(rz_pend);
            if (lane == 0) atomicAdd(rz_acc + b_pend, rz_pend);
        }
#pragma unroll
        for (int k = 0; k < NU; ++k) {
            smooth_step<R, W, T>(xc, c, y0r, y1r, rh0, rh1, (T)ch.w[NU - 1 - k]);
            if (k == 0 && threadIdx.x == 0 && j + 2 < nb) fetch(j + 2);
        }
        double rz = 0.0;
        double* zp = z_out + b * plane + goff;  // (one pointer stepped by the pitch: the per-row form recomputed the 64-bit offset)
#pragma unroll
        for (int i = 0; i < R; ++i) {
            if ((interior >> i) & 1) {
                const float2 s2 = sc_slot[i * 32];
                st2(zp, make_double2((double)((T)s2.x * y0r[i]), (double)((T)s2.y * y1r[i])));
                if (DOT) {  // r.z = r.(s y) = (s r).y = r^.y
                    rz = fma((double)rh0[i], (double)y0r[i], rz);
                    rz = fma((double)rh1[i], (double)y1r[i], rz);
                }
            }
            zp += L.pitch;
        }
        rz_pend = rz;
        b_pend = b;
    }
    if (DOT && b_pend >= 0) {
        rz_pend = warp_sum(rz_pend);
        if (lane == 0) atomicAdd(rz_acc + b_pend, rz_pend);
    }
}

// ---------------------------------------------------------------------------------------------
// Operator apply of the CG iteration (level 0), on the UNSCALED operator (this is the matrix CG solves with, so it
// uses the raw conductances), with the direction kept implicit:
//   w = L z = d z - sum_nb g_nb z_nb ;  q = w + beta q_old   (= L p for p = z + beta p_old, by linearity) ;
//   zw += z.w ;  sumz += sum(z)
// The search direction p itself is never stored: CG needs it only at the port nodes (x_port += alpha p[port]; pcg.cuh
// keeps p[port] = z[port] + beta p_old[port]) and in the scalars p.Lp = z.w - beta^2 p_old.Lp_old (L-conjugacy of
// consecutive directions) and sum(p) = sum(z) + beta sum(p_old) (k_scal_alpha).  That is one vector written and one
// read per iteration less than the textbook update (3 V instead of 4 V).  q is updated in place: a block reads and
// writes q only at its own interior nodes.
// Shared memory: z tiles in two stages (refilled after the apply, as in the V-cycle kernels), q tiles in a ring of
// three (a q tile is consumed at the END of its iteration, so its slot is refilled one iteration later, with the
// right-hand side three ahead: the same two iterations of prefetch lead as z).
template <int R, int W>
__global__ void __launch_bounds__(32 * W, 1)
k_pq3(const __grid_constant__ CUtensorMap tm_z, const __grid_constant__ CUtensorMap tm_q, Level L,
      const double* __restrict__ beta, double* __restrict__ q, double* __restrict__ zw_acc,
      double* __restrict__ sumz_acc, int B, int G, const int* __restrict__ active,
      int first) {  // first: beta = 0 for every right-hand side, q_old is not fetched (it does not exist yet)
    constexpr int H = 2;  // one ring is needed; two keep the 16-byte column pairs aligned
    using Gm = Geom<R, W, H>;
    extern __shared__ __align__(128) double smem_dyn[];
    double* zbuf = smem_dyn;             // 2 stages
    double* qbuf = zbuf + 2 * Gm::TILE;  // 3 slots
    Exch<W>& x = *reinterpret_cast<Exch<W>*>(qbuf + 3 * Gm::TILE);
    __shared__ uint64_t mbar[3];  // two z stages + the row-exchange barrier
    __shared__ uint64_t mbq[3];   // the q ring

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int x0 = blockIdx.x * Gm::IW - H, y0 = blockIdx.y * Gm::IH - H;
    const int gx = x0 + 2 * lane, gy0 = y0 + R * warp;
    const int slot0 = (R * warp) * T3_EW + 2 * lane;
    Patch<R> c;
    patch_init<R, double>(c, L.gx, L.gy, nullptr, L, gx, gy0, nullptr, 0);
    const double zero[R] = {};
    double d0[R], d1[R];  // diagonal = sum of the incident conductances
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const double n0 = i == 0 ? c.hN0 : c.hS0[i == 0 ? 0 : i - 1], n1 = i == 0 ? c.hN1 : c.hS1[i == 0 ? 0 : i - 1];
        d0[i] = (c.hE0[i] + c.hW0[i]) + (c.hS0[i] + n0);
        d1[i] = (c.hE1[i] + c.hE0[i]) + (c.hS1[i] + n1);
    }
    exch_clear<R, W, double>(x);
    const unsigned interior = interior_mask<R, H, Gm::IW, Gm::IH>(L, lane, warp, gx, gy0);
    const size_t plane = (size_t)L.ny * L.pitch;
    const size_t goff = (size_t)gy0 * L.pitch + gx;
    __shared__ ActiveList al;
    active_list_build(al, active, blockIdx.z * G, min(G, B - (int)blockIdx.z * G), beta);
    if (threadIdx.x == 0) {
        mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); mbar_init(&mbar[2], 32 * W);
        mbar_init(&mbq[0], 1); mbar_init(&mbq[1], 1); mbar_init(&mbq[2], 1);
        mbar_fence_init();
    }
    __syncthreads();
    const int nb = al.n;
    auto fetch_z = [&](int j) {  // thread 0 only
        const int st = j & 1;
        mbar_expect_tx(&mbar[st], Gm::TILE_BYTES);
        tma_load_3d(zbuf + st * Gm::TILE, &tm_z, x0, y0, al.b[j], &mbar[st]);
    };
    auto fetch_q = [&](int j) {  // thread 0 only
        const int sq = j % 3;
        mbar_expect_tx(&mbq[sq], Gm::TILE_BYTES);
        tma_load_3d(qbuf + sq * Gm::TILE, &tm_q, x0, y0, al.b[j], &mbq[sq]);
    };
    if (threadIdx.x == 0 && nb > 0) {  // nb == 0: every right-hand side of the group has converged
        fetch_z(0);
        if (nb > 1) fetch_z(1);
        if (!first)
            for (int j = 0; j < 3 && j < nb; ++j) fetch_q(j);
    }
    Xchg<W> xc{&x, &mbar[2], 0, 0u, warp, lane};
    double zw_pend = 0.0, sumz_pend = 0.0;  // partials of the previous right-hand side, reduced one iteration later
    int b_pend = -1;
    auto flush = [&] {
        zw_pend = warp_sum(zw_pend);
        sumz_pend = warp_sum(sumz_pend);
        if (lane == 0) {
            atomicAdd(zw_acc + b_pend, zw_pend);
            atomicAdd(sumz_acc + b_pend, sumz_pend);
        }
    };
    for (int j = 0; j < nb; ++j) {
        const int b = al.b[j], st = j & 1, sq = j % 3;
        mbar_wait(&mbar[st], (j >> 1) & 1);
        const double bt = al.s[j];
        double z0[R], z1[R], sumz = 0.0, zw = 0.0;
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 zz = ld2(zbuf + st * Gm::TILE + slot0 + i * T3_EW);
            sumz += ((interior >> i) & 1) ? zz.x + zz.y : 0.0;
            z0[i] = zz.x;
            z1[i] = zz.y;
        }
        if (b_pend >= 0) flush();
        double t0[R], t1[R];
        apply_step<R, W, double>(xc, c, z0, z1, zero, zero, t0, t1);
        // past this exchange every thread has read its z tile of this iteration and its q tile of the previous one
        if (threadIdx.x == 0 && j + 2 < nb) {
            fetch_z(j + 2);
            if (!first && j >= 1) fetch_q(j + 2);  // slot (j+2) % 3 = (j-1) % 3
        }
        if (!first) mbar_wait(&mbq[sq], (j / 3) & 1);
        double* qp = q + b * plane + goff;
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const bool in = (interior >> i) & 1;
            const double w0 = fma(d0[i], z0[i], -t0[i]), w1 = fma(d1[i], z1[i], -t1[i]);
            double q0 = w0, q1 = w1;
            if (!first) {
                const double2 qo = ld2(qbuf + sq * Gm::TILE + slot0 + i * T3_EW);
                q0 = fma(bt, qo.x, w0);
                q1 = fma(bt, qo.y, w1);
            }
            if (in) st2(qp, make_double2(q0, q1));
            qp += L.pitch;
            zw = fma(in ? z0[i] : 0.0, w0, zw);
            zw = fma(in ? z1[i] : 0.0, w1, zw);
        }
        zw_pend = zw;
        sumz_pend = sumz;
        b_pend = b;
    }
    if (b_pend >= 0) flush();
}

// ---------------------------------------------------------------------------------------------
// The operator apply of an iteration that is EXPECTED TO BE THE LAST of its batch (the host predicts the next residual
// from the contraction so far).  Such an iteration needs neither q nor the new residual as vectors -- only
//   alpha = rho / p.Lp  (for the update of x at the port nodes)   and   ||r - alpha q||^2  (to confirm convergence),
// and the second is a quadratic in alpha whose coefficients do not depend on it:
//   ||r - alpha q||^2 = ||r||^2 - 2 alpha r.q + alpha^2 ||q||^2,    q = L z + beta q_old.
// So this variant reads z, q_old and r (3 V), forms q in registers and reduces z.Lz, sum(z), ||q||^2 and r.q; nothing is
// written.  k_pq3 + the norm probe moved 5 V for the same outcome.  k_scal_estimate turns the sums into ||r_new||^2
// (with a bound on the cancellation error: an estimate it cannot vouch for counts as "not converged"); if the batch
// has not converged after all, the host runs the ordinary k_pq3 and the residual update and carries on.
// q_old and r are needed at the block's interior nodes only: they come as 60 x 68 boxes (their own tensor maps), two
// stages each, refilled one iteration after their use (they are consumed at the end of an iteration).
template <int R, int W>
__global__ void __launch_bounds__(32 * W, 1)
k_pq3_last(const __grid_constant__ CUtensorMap tm_z, const __grid_constant__ CUtensorMap tm_qi,
           const __grid_constant__ CUtensorMap tm_ri, Level L, const double* __restrict__ beta,
           double* __restrict__ zw_acc, double* __restrict__ sumz_acc, double* __restrict__ qq_acc,
           double* __restrict__ rq_acc, int B, int G, const int* __restrict__ active, int first) {
    constexpr int H = 2;
    using Gm = Geom<R, W, H>;
    constexpr int ITILE = Gm::IW * Gm::IH;
    constexpr uint32_t ITILE_BYTES = ITILE * sizeof(double);
    static_assert(ITILE_BYTES % 128 == 0, "TMA destinations are 128-byte aligned");
    extern __shared__ __align__(128) double smem_dyn[];
    double* zbuf = smem_dyn;              // 2 stages, tile + halo
    double* qbuf = zbuf + 2 * Gm::TILE;   // 2 stages, interior only
    double* rbuf = qbuf + 2 * ITILE;      // 2 stages, interior only
    Exch<W>& x = *reinterpret_cast<Exch<W>*>(rbuf + 2 * ITILE);
    __shared__ uint64_t mbar[3];  // two z stages + the row-exchange barrier
    __shared__ uint64_t mbi[2];   // the (q_old, r) stages

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int x0 = blockIdx.x * Gm::IW - H, y0 = blockIdx.y * Gm::IH - H;
    const int gx = x0 + 2 * lane, gy0 = y0 + R * warp;
    const int slot0 = (R * warp) * T3_EW + 2 * lane;
    const int islot0 = (R * warp - H) * Gm::IW + 2 * lane - H;  // the same node in an interior-only tile
    Patch<R> c;
    patch_init<R, double>(c, L.gx, L.gy, nullptr, L, gx, gy0, nullptr, 0);
    const double zero[R] = {};
    double d0[R], d1[R];  // diagonal = sum of the incident conductances
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const double n0 = i == 0 ? c.hN0 : c.hS0[i == 0 ? 0 : i - 1], n1 = i == 0 ? c.hN1 : c.hS1[i == 0 ? 0 : i - 1];
        d0[i] = (c.hE0[i] + c.hW0[i]) + (c.hS0[i] + n0);
        d1[i] = (c.hE1[i] + c.hE0[i]) + (c.hS1[i] + n1);
    }
    exch_clear<R, W, double>(x);
    const unsigned interior = interior_mask<R, H, Gm::IW, Gm::IH>(L, lane, warp, gx, gy0);
    __shared__ ActiveList al;
    active_list_build(al, active, blockIdx.z * G, min(G, B - (int)blockIdx.z * G), beta);
    if (threadIdx.x == 0) {
        mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); mbar_init(&mbar[2], 32 * W);
        mbar_init(&mbi[0], 1); mbar_init(&mbi[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    const int nb = al.n;
    auto fetch_z = [&](int j) {  // thread 0 only
        const int st = j & 1;
        mbar_expect_tx(&mbar[st], Gm::TILE_BYTES);
        tma_load_3d(zbuf + st * Gm::TILE, &tm_z, x0, y0, al.b[j], &mbar[st]);
    };
    auto fetch_i = [&](int j) {  // thread 0 only
        const int st = j & 1;
        mbar_expect_tx(&mbi[st], (first ? 1 : 2) * ITILE_BYTES);
        tma_load_3d(rbuf + st * ITILE, &tm_ri, x0 + H, y0 + H, al.b[j], &mbi[st]);
        if (!first) tma_load_3d(qbuf + st * ITILE, &tm_qi, x0 + H, y0 + H, al.b[j], &mbi[st]);
    };
    if (threadIdx.x == 0 && nb > 0) {  // nb == 0: every right-hand side of the group has converged
        fetch_z(0); fetch_i(0);
        if (nb > 1) { fetch_z(1); fetch_i(1); }
    }
    Xchg<W> xc{&x, &mbar[2], 0, 0u, warp, lane};
    double pend[4] = {0.0, 0.0, 0.0, 0.0};  // partials of the previous right-hand side, reduced one iteration later
    int b_pend = -1;
    auto flush = [&] {
#pragma unroll
        for (int k = 0; k < 4; ++k) pend[k] = warp_sum(pend[k]);
        if (lane == 0) {
            atomicAdd(zw_acc + b_pend, pend[0]);
            atomicAdd(sumz_acc + b_pend, pend[1]);
            atomicAdd(qq_acc + b_pend, pend[2]);
            atomicAdd(rq_acc + b_pend, pend[3]);
        }
    };
    for (int j = 0; j < nb; ++j) {
        const int b = al.b[j], st = j & 1;
        mbar_wait(&mbar[st], (j >> 1) & 1);
        const double bt = al.s[j];
        double z0[R], z1[R], sumz = 0.0, zw = 0.0, qq = 0.0, rq = 0.0;
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 zz = ld2(zbuf + st * Gm::TILE + slot0 + i * T3_EW);
            sumz += ((interior >> i) & 1) ? zz.x + zz.y : 0.0;
            z0[i] = zz.x;
            z1[i] = zz.y;
        }
        if (b_pend >= 0) flush();
        double t0[R], t1[R];
        apply_step<R, W, double>(xc, c, z0, z1, zero, zero, t0, t1);
        // past this exchange every thread has read its z tile of this iteration and its (q_old, r) tiles of the previous one
        if (threadIdx.x == 0) {
            if (j + 2 < nb) fetch_z(j + 2);
            if (j >= 1 && j + 1 < nb) fetch_i(j + 1);  // stage (j+1) & 1 = (j-1) & 1
        }
        mbar_wait(&mbi[st], (j >> 1) & 1);
#pragma unroll
        for (int i = 0; i < R; ++i) {
            if ((interior >> i) & 1) {
                const double w0 = fma(d0[i], z0[i], -t0[i]), w1 = fma(d1[i], z1[i], -t1[i]);
                const double2 rr = ld2(rbuf + st * ITILE + islot0 + i * Gm::IW);
                double q0 = w0, q1 = w1;
                if (!first) {
                    const double2 qo = ld2(qbuf + st * ITILE + islot0 + i * Gm::IW);
                    q0 = fma(bt, qo.x, w0);
                    q1 = fma(bt, qo.y, w1);
                }
                zw = fma(z0[i], w0, zw); zw = fma(z1[i], w1, zw);
                qq = fma(q0, q0, qq);    qq = fma(q1, q1, qq);
                rq = fma(rr.x, q0, rq);  rq = fma(rr.y, q1, rq);
            }
        }
        pend[0] = zw; pend[1] = sumz; pend[2] = qq; pend[3] = rq;
        b_pend = b;
    }
    if (b_pend >= 0) flush();
}

}  // namespace pdn
