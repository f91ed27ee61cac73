// C-ABI entry points (include/pdn.h) and host-side orchestration of the hot path:
//   pdn_create = S0 (tier import + multigrid hierarchy) -> S1 (batched port reduction by MG-PCG)
//                -> S2 (assemble C) -> S3 (factor once, substitute for m+n right-hand sides)
//   pdn_reff   = S4 (pair evaluation) [+ S5 copy to host]
// Everything numerical runs in the kernels of stencil3.cuh / tail.cuh / pcg.cuh / setup.cuh / uniform.cuh /
// dense.cuh / port.cuh; the host code (host_runtime.cuh: pool, context, launch bookkeeping; host_solve.cuh:
// hierarchy, workspace, V-cycle, batched PCG loop; host_recombine.cuh: S2 + S3; this file: the entry points)
// only validates, allocates, encodes TMA descriptors, sequences launches and reads back the per-batch
// convergence counters.  There is no CPU fallback.
#include "../../include/pdn.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <thread>
#include <new>
#include <set>
#include <string>
#include <utility>
#include <vector>

#include "common.cuh"
#include "dense.cuh"
#include "pcg.cuh"
#include "port.cuh"
#include "setup.cuh"
#include "stencil3.cuh"
#include "tail.cuh"
#include "uniform.cuh"
#include "guess.cuh"
#include "host_runtime.cuh"
#include "host_solve.cuh"
#include "host_recombine.cuh"

namespace {

// ------------------------------------------------------------------------------------------------
// Host-side pieces shared by pdn_create and pdn_update_tsvs.

// Validates a TSV list and splits it per interface (sites as pitched offsets y*pitch + x, in list order).
void parse_tsvs(int d, int n, int n_tsv, const pdn_tsv* tsvs, std::vector<std::vector<int>>& site,
                std::vector<std::vector<double>>& rt) {
    site.assign(d - 1, {});
    rt.assign(d - 1, {});
    std::vector<std::set<int>> seen(d - 1);
    for (int k = 0; k < n_tsv; ++k) {
        const pdn_tsv& t = tsvs[k];
        if (t.iface < 0 || t.iface >= d - 1) throw StatusFail{PDN_E_ARG, "TSV interface out of range"};
        if (t.y < 0 || t.y >= n || t.x < 0 || t.x >= n) throw StatusFail{PDN_E_ARG, "TSV site out of range"};
        if (!(t.r_ohm > 0.0) || !std::isfinite(t.r_ohm)) throw StatusFail{PDN_E_ARG, "TSV resistance must be positive and finite"};
        const int id = t.y * pitch_of(n) + t.x;  // pitched offset (port.cuh / pcg.cuh index vectors with it)
        if (!seen[t.iface].insert(id).second) throw StatusFail{PDN_E_ARG, "duplicate TSV site inside one interface"};
        site[t.iface].push_back(id);
        rt[t.iface].push_back(t.r_ohm);
    }
    for (int i = 0; i < d - 1; ++i)
        if (site[i].empty()) throw StatusFail{PDN_E_ARG, "an interface has no TSV"};
}

// Port list of tier t:  [lower ends of interface t-1] ++ [upper ends of interface t] ++ [terminals].
void tier_port_list(const pdn_ctx* c, int t, const std::vector<std::vector<int>>& site, std::vector<int>& node, int& ntsv) {
    node.clear();
    if (t > 0) node.insert(node.end(), site[t - 1].begin(), site[t - 1].end());
    if (t < c->d - 1) node.insert(node.end(), site[t].begin(), site[t].end());
    ntsv = (int)node.size();
    if (t == 0) node.insert(node.end(), c->bump_id.begin(), c->bump_id.end());
    if (c->d == 1) ntsv = (int)node.size();  // single tier: the bumps are the row sources, the loads the terminals
    if (t == c->d - 1) node.insert(node.end(), c->load_id.begin(), c->load_id.end());
}

// Right-hand sides per batch: what fits in 60 % of the free device memory (pool blocks count as free).
int pick_batch(const Hierarchy& H, int want, const pdn_opts& o) {
    if (H.nlev <= 1) return std::max(want, 1);
    size_t free_b = 0, total_b = 0;
    CK(cudaMemGetInfo(&free_b, &total_b));
    free_b += g_pool.cached_bytes(DevPool::current_device());
    const size_t per = Work::bytes_per_rhs(H) + (size_t)want * 8 + 128;
    const size_t fit = std::max<size_t>(1, (size_t)(0.6 * (double)free_b) / per);
    int B = (int)std::min<size_t>({(size_t)std::max(want, 1), fit, (size_t)1024});
    if (o.rhs_batch > 0) B = std::min(B, o.rhs_batch);
    return B;
}

// Spectral tables of Eq. (3) (uniform.cuh) built during one call, keyed by mesh size and rho = g_x / g_y: tiers that
// differ by a scale factor share a table (a uniform stack builds one table, not one per tier; the initial guess of
// BASELINE's workloads builds one per call).
struct SpectralTables {
    struct Entry { int n; double rho; DevBuf G, Gf, Gq; CUtensorMap map_q; };  // Gq: FP32, pitched, behind map_q
    std::vector<Entry> list;
    Entry* find(int n, double rho, double rel_tol) {
        for (Entry& e : list)
            if (e.n == n && std::fabs(e.rho - rho) <= rel_tol * rho) return &e;
        return nullptr;
    }
    Entry& build(Launcher& L, int n, double rho, bool want_float) {
        const size_t nn = (size_t)n * n, n1 = (size_t)n + 1;
        Entry e;
        e.n = n; e.rho = rho;
        e.G.alloc(n1 * n1 * sizeof(double));
        DevBuf Cm, Wm, T1;
        Cm.alloc(n1 * n * sizeof(double)); Wm.alloc(nn * sizeof(double)); T1.alloc(n * n1 * sizeof(double));
        L.run(KC_SMALL, 0, [&] { k_cos_matrix<<<cdiv(n1 * n, 256), 256, 0, L.s>>>(n, Cm.as<double>()); });
        L.run(KC_SMALL, 0, [&] { k_spectral_weights<<<cdiv(nn, 256), 256, 0, L.s>>>(n, rho, 1.0, Wm.as<double>()); });
        // T[a][s] = sum_b W[a][b] C[s][b]  (n x (n+1));  G[t][s] = sum_a C[t][a] T[a][s]  ((n+1) x (n+1))
        gemm(L, n, n + 1, n, 1.0, Wm.as<double>(), n, 1, Cm.as<double>(), 1, n, 0.0, T1.as<double>(), n + 1);
        gemm(L, n + 1, n + 1, n, 1.0, Cm.as<double>(), n, 1, T1.as<double>(), n + 1, 1, 0.0, e.G.as<double>(), n + 1);
        CK(cudaStreamSynchronize(L.s));  // the work buffers go back to the pool here
        list.push_back(std::move(e));
        Entry& r = list.back();
        if (want_float) float_copy(L, r);
        return r;
    }
    void float_copy(Launcher& L, Entry& e) {
        if (e.Gf.p) return;
        const size_t cnt = ((size_t)e.n + 1) * (e.n + 1);
        e.Gf.alloc(cnt * sizeof(float));
        const int pq = (e.n + 1 + 3) & ~3;
        e.Gq.alloc((size_t)(e.n + 1) * pq * sizeof(float));
        L.run(KC_SMALL, 0, [&] { k_table_to_float<<<cdiv(cnt, 256), 256, 0, L.s>>>(cnt, e.G.as<double>(), e.Gf.as<float>()); });
        L.run(KC_SMALL, 0, [&] { k_table_to_pitched<<<cdiv((size_t)(e.n + 1) * pq, 256), 256, 0, L.s>>>(e.n, pq, e.G.as<double>(), e.Gq.as<float>()); });
        e.map_q = make_map_2d_f32(e.Gq.p, e.n + 1, e.n + 1, pq, GW_BW, GuessRhsGeom::BH);
    }
};

// S1 of one tier whose hierarchy H has just been built: fills rows `tsv_src` of ZT (each against all ports of
// the tier) and, if `terminals`, zdiag.  Meshes with n <= 4 and uniform tiers (Eq. 3) are reduced whole.
int reduce_tier(pdn_ctx* c, Launcher& L, Hierarchy& H, Work& W, int Bmax, TierPorts& T, const std::vector<int>& tsv_src,
                const std::vector<int>& term, SpectralTables& tabs,  // term: port indices (>= ntsv) of the terminal sources to solve
                bool diag_only_terms = false) {                      // ... for their diagonal only, whatever PDN_TERMINAL_PAIRS says
    T.whole = false;
    const pdn_opts& o = c->opts;
    const int n = c->n;
    if (H.nlev == 1) {
        L.run(KC_SMALL, 0, [&] { k_direct_small<<<T.q, 64, 0, L.s>>>(H.pinv.as<double>(), n, H.pitch[0], n * n, T.d_node.as<int>(), T.ntsv, T.nrows, T.q, T.ZT.as<double>(), T.zdiag.as<double>()); });
        T.whole = true;
        return PDN_OK;
    }
    // The spectral table of a uniform tier costs 4 n^3 flops whatever the port count; q port solves cost about
    // 8 iterations x 14 passes over a vector each.  With few ports on a very large mesh the solves are cheaper,
    // so the table is used only where this model says it pays -- or where an earlier tier of the call left one
    // (FP64 tensor-core rate of the two contractions: ~3 TF/s at n = 1024, saturating near 22 TF/s).
    const double nn = (double)n * n;
    const double t_table = 1e-4 + 4.0 * nn * n / std::min(22e12, 3e12 * n / 1024.0);
    const double t_solves = 5e-4 + (double)T.q * 112.0 * 8.0 * nn / 4e12;
    if (!(o.flags & PDN_NO_UNIFORM_FAST_PATH) && H.cv <= 1e-6) {
        // uniform tier: Eq. (3) of the paper as two dense contractions + a gather (uniform.cuh)
        int* fl = H.flags.as<int>();
        CK(cudaMemsetAsync(fl, 0, sizeof(int), L.s));
        L.run(KC_SMALL, 0, [&] { k_uniform_check<<<cdiv(H.plane(0), 256), 256, 0, L.s>>>(n, H.pitch[0], H.gx[0].as<double>(), H.gy[0].as<double>(), fl); });
        int h_flag = 1;
        double g0[2] = {0.0, 0.0};
        CK(cudaMemcpyAsync(&h_flag, fl, sizeof(int), cudaMemcpyDeviceToHost, L.s));
        CK(cudaMemcpyAsync(&g0[0], H.gx[0].p, sizeof(double), cudaMemcpyDeviceToHost, L.s));
        CK(cudaMemcpyAsync(&g0[1], H.gy[0].p, sizeof(double), cudaMemcpyDeviceToHost, L.s));
        CK(cudaStreamSynchronize(L.s));
        if (h_flag == 0 && g0[0] > 0.0 && g0[1] > 0.0) {
            const double rho = g0[0] / g0[1];
            SpectralTables::Entry* e = tabs.find(n, rho, 0.0);
            if (!e && t_table <= t_solves) e = &tabs.build(L, n, rho, false);
            if (e) {
                L.run(KC_SMALL, 0, [&] { k_uniform_gather<<<dim3(cdiv(T.q, 128), grid_rows((size_t)T.nrows + 1)), 128, 0, L.s>>>(e->G.as<double>(), 1.0 / g0[1], n, H.pitch[0], T.d_node.as<int>(), T.ntsv, T.nrows, T.q, T.ZT.as<double>(), T.zdiag.as<double>()); });
                { std::lock_guard<std::mutex> g(c->mu); c->stats.n_uniform_tiers++; }
                T.whole = true;
                return PDN_OK;
            }
        }
    }
    // Initial guess (guess.cuh): the closed form of the tier's MEAN mesh as the starting point of every port solve,
    // where the tier is near enough to it (coefficient of variation of the segment conductances; a rejected guess
    // costs one pass over the vector) and large enough for an iteration to be worth more than the extra launches.
    // A table left by an earlier tier of the call with the same anisotropy (within 2 %) is reused: the guess need
    // not be exact.  A new one is built only for enough right-hand sides to pay for its 4 n^3 flops.
    GuessHost gtab{};
    const GuessHost* guess = nullptr;
    if (!(o.flags & PDN_NO_INITIAL_GUESS) && n >= 192 && H.cv <= 0.5 && H.mean_gx > 0.0 && H.mean_gy > 0.0) {
        const double rho = H.mean_gx / H.mean_gy;
        SpectralTables::Entry* e = tabs.find(n, rho, 0.02);
        if (!e && (long)(tsv_src.size() + term.size()) >= n / 2) e = &tabs.build(L, n, rho, true);
        if (e) {
            tabs.float_copy(L, *e);
            gtab = GuessHost{GuessTable{e->Gf.as<float>(), 1.0 / H.mean_gy, n}, e->map_q};
            guess = &gtab;
            { std::lock_guard<std::mutex> g(c->mu); c->stats.n_guess_tiers++; }
        }
    }
    // Smoothing interval [2/ratio, 2] of the Chebyshev polynomial.  With 2x2 aggregation the coarse grid
    // takes fewer modes off the smoother the more anisotropic the tier is, so the interval widens with
    // the anisotropy a: ratio = 3 + a (measured: a = 1 -> 4, a = 3 -> 6).
    // Strongly anisotropic tiers (a >= 6) leave modes that are smooth along the strong direction and oscillatory
    // across it, with eigenvalues down to ~2/(1+a) of D^-1 L, to the smoother: the interval becomes [1/(1+a), 2]
    // and, unless the caller fixed nu, the smoother gets the deepest polynomial the kernels have (measured at
    // 512^2: a = 10 / 30 / 100 need 9 / 12 / 40 iterations this way against 16 / 62 / 146 with the rule above).
    const bool strong = H.anisotropy >= 6.0;
    const int nu = (strong && c->nu_auto) ? 6 : o.nu;
    const double ratio = o.cheb_ratio > 1.0 ? o.cheb_ratio : strong ? 2.0 * (1.0 + H.anisotropy) : 3.0 + H.anisotropy;
    const int G = T3_MAX_G;  // upper bound of the right-hand sides a stencil block loops over (rhs_per_block picks)
    // On near-isotropic tiers the coarse levels get by with one step less on a wider interval (measured: same
    // iteration counts at configs 3 and 5, one level-visit cheaper); anisotropic tiers keep nu steps everywhere.
    const bool iso = H.anisotropy < 1.5 && nu >= 3 && !(o.cheb_ratio > 1.0);
    const int nu_c = iso ? nu - 1 : nu;
    const double ratio_c = iso ? 2.0 * ratio : ratio;
    const bool f32 = (o.flags & PDN_PRECOND_F32) != 0;
    const Smoother ch{make_cheb_roots(nu, ratio), make_cheb_roots(nu_c, ratio_c), G, f32};
    // bump / load sources deliver only their own diagonal, whose CG error is the square of the energy-norm error
    // (times the condition number of the preconditioned operator, which is why a caller who tightens rtol below
    // the default also gets tighter terminal solves: at most 1000 rtol)
    const double rtol_term = std::max(o.rtol, std::min({1e-5, std::sqrt(o.rtol) / 3.0, 1e3 * o.rtol}));
    int status = PDN_OK;
    for (size_t s0 = 0; s0 < tsv_src.size() && status == PDN_OK; s0 += Bmax)
        status = solve_batch(c, L, H, W, T, ch, tsv_src.data() + s0, (int)std::min<size_t>(Bmax, tsv_src.size() - s0), false, o.rtol, o.max_iter, guess);
    if (!term.empty()) {
        // with the terminal rows kept they are ordinary rows of ZT: full tolerance, gathered at every port
        const bool rows = c->terminal_pairs && !diag_only_terms;
        for (size_t s0 = 0; s0 < term.size() && status == PDN_OK; s0 += Bmax)
            status = solve_batch(c, L, H, W, T, ch, term.data() + s0, (int)std::min<size_t>(Bmax, term.size() - s0), !rows,
                                 rows ? o.rtol : rtol_term, o.max_iter, guess);
        if (rows && status == PDN_OK && !c->open)  // (an open, sharded context does this in pdn_finish)
            L.run(KC_SMALL, 0, [&] { k_zdiag_from_rows<<<cdiv(T.nterm, 128), 128, 0, L.s>>>(T.ZT.as<double>(), T.q, T.ntsv, T.nterm, T.zdiag.as<double>()); });
    }
    return status;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// pdn_load_voltages_static: Eq. (4) without any allocation.  pdn_load_voltages takes its scratch (R_b: n values,
// R_LL: n x n values, two index lists) from the device pool, which calls cudaMalloc when the pool has no block of
// that size.  This variant keeps the scratch in the file-scope array below -- part of the library's image: every GPU
// that loads libpdn.so holds these 2.0 MiB until the process exits -- for at most PDN_STATIC_MAX_LOADS loads.
//   layout: R_LL at [0, n*n), R_b at [MAXL*MAXL, MAXL*MAXL + n)   (both 256-byte aligned)
// Every word a call reads was written earlier by the same call (k_pair_same writes all n*n entries of R_LL,
// k_pair_row all n of R_b): nothing has to start at zero and what the previous call left is never read.  All calls on
// one device share the array: two calls whose kernels overlap on the GPU (two contexts on different streams, two host
// threads) race.
// In host code `g_static_scratch` is the host-side shadow of the symbol, NOT a device address: the kernels get the
// pointer cudaGetSymbolAddress returns, resolved once per device with that device current.
constexpr int STATIC_MAXL = PDN_STATIC_MAX_LOADS;
static __device__ __align__(256) double g_static_scratch[(size_t)STATIC_MAXL * STATIC_MAXL + STATIC_MAXL];

static double* static_scratch_of_current_device() {
    static std::mutex mu;
    static double* ptr[64] = {};
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) throw StatusFail{PDN_E_ARG, "device ordinal out of range"};
    std::lock_guard<std::mutex> g(mu);
    if (!ptr[dev]) {
        double* p = nullptr;
        CK(cudaGetSymbolAddress((void**)&p, g_static_scratch));
        if (!p || ((uintptr_t)p & 255)) throw StatusFail{PDN_E_CUDA, "static scratch array has no usable device address"};
        ptr[dev] = p;
    }
    return ptr[dev];
}

// R_b[j] = R_eff(bump i, load j) for all loads: k_pair_list on the pairs (i, 0..n-1) without index lists in memory
// (same loop, same association: the same bits).  One warp per load.
__global__ void k_pair_row(int i, int n, int p0, const double* __restrict__ A1, const double* __restrict__ X0,
                           const double* __restrict__ u, const double* __restrict__ w, double* __restrict__ R) {
    const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (j >= n) return;
    double s = 0.0;
    for (int a = lane; a < p0; a += 32) s = fma(A1[(int64_t)i * p0 + a], X0[(int64_t)j * p0 + a], s);
    s = warp_sum(s);
    if (lane == 0) R[j] = u[i] + w[j] - 2.0 * s;
}

// ================================================================================================
// C ABI
// ================================================================================================
extern "C" {

const char* pdn_strerror(int status) {
    switch (status) {
        case PDN_OK: return "ok";
        case PDN_E_ARG: return "invalid argument";
        case PDN_E_DISCONNECTED: return "a tier is not connected";
        case PDN_E_NOCONV: return "port solve did not converge within max_iter";
        case PDN_E_CUDA: return "CUDA error";
        case PDN_E_NOMEM: return "out of memory";
        case PDN_E_NUMERIC: return "port-level matrix not positive definite";
        default: return "unknown status";
    }
}

const char* pdn_last_error(void) { return g_last_error.c_str(); }

void pdn_destroy(pdn_ctx* ctx) {
    if (!ctx) return;
    for (cudaEvent_t e : ctx->event_pool) cudaEventDestroy(e);
    for (auto& pe : ctx->pending_events) { cudaEventDestroy(pe.second.first); cudaEventDestroy(pe.second.second); }
    delete ctx;
}

static int fail_arg(const char* msg) {
    g_last_error = msg;
    return PDN_E_ARG;
}

// A context lives on the device that was current at pdn_create; every later call must be made with it current.
static bool wrong_device(const pdn_ctx* c) {
    int dev = -1;
    return cudaGetDevice(&dev) != cudaSuccess || dev != c->device;
}
#define PDN_CHECK_DEVICE(ctx)                                                                                      \
    do {                                                                                                           \
        if ((ctx)->poisoned) return fail_arg("the context is unusable after a failed pdn_update_tsvs: destroy it"); \
        if (wrong_device(ctx)) return fail_arg("the context's CUDA device is not the current device");             \
    } while (0)

int pdn_create(pdn_ctx** out, int32_t n_tiers, const pdn_tier* tiers, int32_t n_tsv, const pdn_tsv* tsvs,
               int32_t n_bumps, const pdn_site* bumps, int32_t n_loads, const pdn_site* loads, const pdn_opts* opts) {
    if (!out) return fail_arg("out is null");
    *out = nullptr;
    if (!tiers || !bumps || !loads || (!tsvs && n_tsv > 0)) return fail_arg("null input array");
    if (n_tiers < 1) return fail_arg("need at least 1 tier");
    if (n_tiers == 1 ? n_tsv != 0 : n_tsv < 1) return fail_arg("need at least one TSV per interface (and none for a single tier)");
    if (n_bumps < 1 || n_loads < 1) return fail_arg("need at least one bump and one load");
    const int d = n_tiers, n = tiers[0].n;
    if (n < 2) return fail_arg("mesh size n must be >= 2");
    if ((int64_t)n * n > (int64_t)1 << 30) return fail_arg("mesh too large");
    for (int t = 0; t < d; ++t) {
        if (tiers[t].n != n) return fail_arg("all tiers must have the same n");
        if (!tiers[t].gx || !tiers[t].gy) return fail_arg("null conductance plane");
    }
    pdn_opts o{};
    if (opts) o = *opts;
    if (!(o.rtol > 0.0)) o.rtol = 1e-8;
    if (o.max_iter <= 0) o.max_iter = 200;
    const bool nu_auto = o.nu <= 0;
    if (o.nu <= 0) o.nu = 4;
    if (o.nu > 6) o.nu = 6;

    pdn_ctx* c = new (std::nothrow) pdn_ctx();
    if (!c) return PDN_E_NOMEM;
    int status = PDN_OK;
    try {
        c->d = d; c->n = n; c->m = n_bumps; c->nl = n_loads; c->opts = o;
        c->stream = (cudaStream_t)o.cuda_stream;
        c->time_kernels = (o.flags & PDN_TIME_KERNELS) != 0;
        c->debug = getenv("PDN_DEBUG") != nullptr;
        c->terminal_pairs = (o.flags & PDN_TERMINAL_PAIRS) != 0;
        c->nu_auto = nu_auto;
        if (o.shard_world > 1) {
            if (d == 1) throw StatusFail{PDN_E_ARG, "sharding needs at least 2 tiers"};
            if (o.shard_rank < 0 || o.shard_rank >= o.shard_world) throw StatusFail{PDN_E_ARG, "shard_rank out of range"};
            c->shard_world = o.shard_world; c->shard_rank = o.shard_rank; c->open = true;
        }
        // ---- host-side validation and port lists
        parse_tsvs(d, n, n_tsv, tsvs, c->site, c->rt);
        c->p.assign(d - 1, 0);
        for (int i = 0; i < d - 1; ++i) c->p[i] = (int)c->site[i].size();
        auto check_sites = [&](const pdn_site* s, int cnt, std::vector<int>& ids) {
            for (int k = 0; k < cnt; ++k) {
                if (s[k].y < 0 || s[k].y >= n || s[k].x < 0 || s[k].x >= n) throw StatusFail{PDN_E_ARG, "bump/load site out of range"};
                ids.push_back(s[k].y * pitch_of(n) + s[k].x);
            }
        };
        check_sites(bumps, n_bumps, c->bump_id);
        check_sites(loads, n_loads, c->load_id);

        CK(cudaGetDevice(&c->device));
        Launcher L{c, c->stream};
        cudaEvent_t ev[4];
        for (auto& e : ev) CK(cudaEventCreate(&e));
        CK(cudaEventRecord(ev[0], L.s));

        c->tiers.resize(d);
        int qmax = 0;
        for (int t = 0; t < d; ++t) {
            TierPorts& T = c->tiers[t];
            tier_port_list(c, t, c->site, T.node, T.ntsv);
            T.q = (int)T.node.size();
            T.nterm = T.q - T.ntsv;
            T.d_node.alloc((size_t)T.q * sizeof(int));
            CK(cudaMemcpyAsync(T.d_node.p, T.node.data(), (size_t)T.q * sizeof(int), cudaMemcpyHostToDevice, L.s));
            T.nrows = (c->terminal_pairs && T.nterm > 0) ? T.q : T.ntsv;
            T.ZT.alloc((size_t)T.nrows * T.q * sizeof(double));
            T.zdiag.alloc((size_t)std::max(T.nterm, 1) * sizeof(double));
            qmax = std::max(qmax, T.q);
            c->stats.n_ports_total += T.q;
        }
        c->stats.n_tiers = d;

        // ---- S0 + S1, tier by tier.  One tier: import + hierarchy (S0), then its port solves (S1).
        std::mutex msg_mu;
        std::string first_msg;
        float ms_up = 0.f;
        auto run_tier = [&](int t, Launcher& TL, Hierarchy& H, Work& W, int Bmax, DevBuf& stage, SpectralTables& tabs,
                            cudaEvent_t e0, cudaEvent_t e1) -> int {
            TierPorts& T = c->tiers[t];
            const double *gx = tiers[t].gx, *gy = tiers[t].gy;
            CK(cudaEventRecord(e0, TL.s));
            if (o.flags & PDN_TIERS_ON_HOST) {
                double* sg = stage.as<double>();
                CK(cudaMemcpyAsync(sg, gx, (size_t)n * n * sizeof(double), cudaMemcpyHostToDevice, TL.s));
                CK(cudaMemcpyAsync(sg + (size_t)n * n, gy, (size_t)n * n * sizeof(double), cudaMemcpyHostToDevice, TL.s));
                gx = sg; gy = sg + (size_t)n * n;
            }
            int st = H.build(TL, gx, gy, !(o.flags & PDN_SKIP_CONNECTIVITY_CHECK));
            if (st == PDN_OK) {  // keep the sanitised planes: pdn_update_tsvs rebuilds the hierarchy from them
                T.gx0.alloc(H.plane(0) * sizeof(double));
                T.gy0.alloc(H.plane(0) * sizeof(double));
                CK(cudaMemcpyAsync(T.gx0.p, H.gx[0].p, H.plane(0) * sizeof(double), cudaMemcpyDeviceToDevice, TL.s));
                CK(cudaMemcpyAsync(T.gy0.p, H.gy[0].p, H.plane(0) * sizeof(double), cudaMemcpyDeviceToDevice, TL.s));
            }
            CK(cudaEventRecord(e1, TL.s));
            CK(cudaEventSynchronize(e1));
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, e0, e1));
            if (st == PDN_OK) {
                // this rank's contiguous slice of the TSV sources and of the terminal sources (everything if unsharded)
                const int W_ = c->shard_world, r_ = c->shard_rank;
                std::vector<int> tsv_src, term_src;
                for (int k = (int)((int64_t)r_ * T.ntsv / W_); k < (int)((int64_t)(r_ + 1) * T.ntsv / W_); ++k) tsv_src.push_back(k);
                for (int k = (int)((int64_t)r_ * T.nterm / W_); k < (int)((int64_t)(r_ + 1) * T.nterm / W_); ++k) term_src.push_back(T.ntsv + k);
                st = reduce_tier(c, TL, H, W, Bmax, T, tsv_src, term_src, tabs);
            }
            std::lock_guard<std::mutex> g(msg_mu);
            ms_up += ms;
            if (st != PDN_OK && first_msg.empty()) {
                const std::string detail = g_last_error;
                first_msg = std::string("tier ") + std::to_string(t) + ": " + pdn_strerror(st) + (detail.empty() ? "" : " (" + detail + ")");
            }
            return st;
        };
        // Small meshes (configs[0..1]: 32^2, 128^2) are bound by the serial latency of many tiny launches, not by the
        // device: their tiers -- independent 2D problems -- are solved concurrently, one host thread
        // and one stream per tier (up to four), each with its own hierarchy and workspace.  Large meshes fill the
        // device with one tier and keep the single-stream path (and one shared spectral table).
        const int n_workers = (n <= 256 && d >= 2) ? std::min(d, 4) : 1;
        c->stats.n_levels = 1;
        for (int cur = n; cur > COARSEST_MAX; cur = (cur + 1) / 2) c->stats.n_levels++;
        if (n_workers == 1) {
            SpectralTables tabs;
            Hierarchy H;
            H.allocate(n);
            DevBuf stage;  // staging for host-resident planes
            if (o.flags & PDN_TIERS_ON_HOST) stage.alloc((size_t)2 * n * n * sizeof(double));
            const int Bmax = pick_batch(H, qmax, o);
            Work W;
            if (H.nlev > 1) W.allocate(H, Bmax, qmax);
            for (int t = 0; t < d && status == PDN_OK; ++t) status = run_tier(t, L, H, W, Bmax, stage, tabs, ev[1], ev[2]);
        } else {
            cudaEvent_t ev_start;
            CK(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
            CK(cudaEventRecord(ev_start, L.s));
            std::vector<int> wst(n_workers, PDN_OK);
            std::vector<cudaEvent_t> ev_done(n_workers, nullptr);
            std::vector<std::thread> th;
            for (int w = 0; w < n_workers; ++w)
                th.emplace_back([&, w] {
                    cudaStream_t ws = nullptr;
                    cudaEvent_t e0 = nullptr, e1 = nullptr;
                    try {
                        CK(cudaSetDevice(c->device));
                        CK(cudaStreamCreateWithFlags(&ws, cudaStreamNonBlocking));
                        CK(cudaStreamWaitEvent(ws, ev_start, 0));
                        CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
                        CK(cudaEventCreateWithFlags(&ev_done[w], cudaEventDisableTiming));
                        Launcher TL{c, ws};
                        SpectralTables tabs;
                        Hierarchy H;
                        H.allocate(n);
                        DevBuf stage;
                        if (o.flags & PDN_TIERS_ON_HOST) stage.alloc((size_t)2 * n * n * sizeof(double));
                        int qw = 1;
                        for (int t = w; t < d; t += n_workers) qw = std::max(qw, c->tiers[t].q);
                        const int Bmax = pick_batch(H, qw, o);
                        Work W;
                        if (H.nlev > 1) W.allocate(H, Bmax, qw);
                        for (int t = w; t < d && wst[w] == PDN_OK; t += n_workers) wst[w] = run_tier(t, TL, H, W, Bmax, stage, tabs, e0, e1);
                        CK(cudaStreamSynchronize(ws));  // the worker's buffers are released when it returns
                        CK(cudaEventRecord(ev_done[w], ws));
                    } catch (const CudaFail& f) {
                        wst[w] = f.e == cudaErrorMemoryAllocation ? PDN_E_NOMEM : PDN_E_CUDA;
                        cudaGetLastError();
                        std::lock_guard<std::mutex> g(msg_mu);
                        if (first_msg.empty()) first_msg = std::string(f.what) + ": " + cudaGetErrorString(f.e);
                    } catch (const StatusFail& f) {
                        wst[w] = f.status;
                        std::lock_guard<std::mutex> g(msg_mu);
                        if (first_msg.empty()) first_msg = f.msg;
                    } catch (const std::bad_alloc&) {
                        wst[w] = PDN_E_NOMEM;
                        std::lock_guard<std::mutex> g(msg_mu);
                        if (first_msg.empty()) first_msg = "host allocation failed";
                    }
                    if (e0) cudaEventDestroy(e0);
                    if (e1) cudaEventDestroy(e1);
                    if (ws) cudaStreamDestroy(ws);
                });
            for (auto& t_ : th) t_.join();
            for (int w = 0; w < n_workers; ++w) {
                if (ev_done[w]) { cudaStreamWaitEvent(L.s, ev_done[w], 0); cudaEventDestroy(ev_done[w]); }
                if (wst[w] != PDN_OK && status == PDN_OK) status = wst[w];
            }
            cudaEventDestroy(ev_start);
        }
        if (status != PDN_OK) g_last_error = first_msg;
        CK(cudaEventRecord(ev[2], L.s));
        // ---- S2 + S3 (a sharded context stays open until its rows are complete: pdn_finish)
        if (status == PDN_OK && !c->open) {
            status = recombine(c, L);
            if (status != PDN_OK) g_last_error = pdn_strerror(status);
        }
        CK(cudaEventRecord(ev[3], L.s));
        CK(cudaStreamSynchronize(L.s));
        L.resolve();
        float ms_all = 0.f, ms_dense = 0.f, ms_s01 = 0.f;
        CK(cudaEventElapsedTime(&ms_all, ev[0], ev[3]));
        CK(cudaEventElapsedTime(&ms_dense, ev[2], ev[3]));
        CK(cudaEventElapsedTime(&ms_s01, ev[0], ev[2]));
        c->stats.ms_total = ms_all; c->stats.ms_dense = ms_dense; c->stats.ms_upload = ms_up;
        c->stats.ms_stencil = ms_s01 - ms_up;
        for (auto& e : ev) cudaEventDestroy(e);
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        status = f.e == cudaErrorMemoryAllocation ? PDN_E_NOMEM : PDN_E_CUDA;
    } catch (const StatusFail& f) {
        g_last_error = f.msg;
        status = f.status;
    } catch (const std::bad_alloc&) {
        g_last_error = "host allocation failed";
        status = PDN_E_NOMEM;
    }
    if (status != PDN_OK) {
        pdn_destroy(c);
        return status;
    }
    *out = c;
    return PDN_OK;
}

// NEXT-2: TSV re-planning.  The new TSV list is diffed against the current one per interface
// by site.  A kept site keeps its rows / columns of the tier port matrices (its resistance may change freely:
// it only enters K); a removed site drops them; an added site costs ONE port solve on each of its two tiers,
// whose solution gives the new row and -- by symmetry of L^+ -- the new column.  C is then re-assembled and
// re-factored (milliseconds).
int pdn_update_tsvs(pdn_ctx* ctx, int32_t n_tsv, const pdn_tsv* tsvs) {
    if (!ctx || !tsvs || n_tsv < 1) return fail_arg("null context / TSV list or empty list");
    PDN_CHECK_DEVICE(ctx);
    if (ctx->open || ctx->shard_world > 1) return fail_arg("TSV re-planning is not available on a sharded context");
    if (ctx->d < 2) return fail_arg("a single-tier context has no TSVs");
    pdn_ctx* c = ctx;
    const int d = c->d, n = c->n;
    int status = PDN_OK;
    bool committed = false;  // the staged tiers were swapped in: a failure after that point poisons the context
    try {
        std::vector<std::vector<int>> nsite;
        std::vector<std::vector<double>> nrt;
        parse_tsvs(d, n, n_tsv, tsvs, nsite, nrt);
        Launcher L{c, c->stream};
        cudaEvent_t ev[3];
        for (auto& e : ev) CK(cudaEventCreate(&e));
        CK(cudaEventRecord(ev[0], L.s));
        // old index -> new index per interface (-1 = removed)
        std::vector<std::vector<int>> o2n(d - 1);
        for (int i = 0; i < d - 1; ++i) {
            std::map<int, int> where;
            for (size_t k = 0; k < nsite[i].size(); ++k) where[nsite[i][k]] = (int)k;
            o2n[i].assign(c->site[i].size(), -1);
            for (size_t k = 0; k < c->site[i].size(); ++k) {
                auto it = where.find(c->site[i][k]);
                if (it != where.end()) o2n[i][k] = it->second;
            }
        }
        SpectralTables tabs;
        Hierarchy H;
        bool h_ready = false;
        int64_t new_solves = 0;
        // Every tier's new port list, port matrix and device copies are built in `staged` and swapped into the
        // context only after ALL tiers succeeded: a failure on a later tier (PDN_E_NOCONV, PDN_E_NOMEM, ...) leaves
        // the context exactly as it was, still valid for the old plan.
        std::vector<TierPorts> staged(d);
        std::vector<char> changed(d, 0);
        for (int t = 0; t < d && status == PDN_OK; ++t) {
            const TierPorts& T = c->tiers[t];
            TierPorts& N = staged[t];
            tier_port_list(c, t, nsite, N.node, N.ntsv);
            if (N.node == T.node) continue;  // same sites in the same order: Z_t is unchanged
            changed[t] = 1;
            const int q_o = T.q, ntsv_o = T.ntsv, q_n = (int)N.node.size(), ntsv_n = N.ntsv;
            const int rows_o = T.nrows, rows_n = (c->terminal_pairs && q_n > ntsv_n) ? q_n : ntsv_n;
            N.q = q_n; N.nterm = q_n - ntsv_n; N.nrows = rows_n;
            const int plo_o = t > 0 ? (int)c->site[t - 1].size() : 0, plo_n = t > 0 ? (int)nsite[t - 1].size() : 0;
            std::vector<int> cmap(q_o, -1);
            std::vector<unsigned char> is_added(std::max(rows_n, 1), 0);
            for (int k = 0; k < ntsv_n; ++k) is_added[k] = 1;
            for (int k = 0; k < ntsv_o; ++k) {
                int kn = -1;
                if (k < plo_o) kn = o2n[t - 1][k];
                else { const int m = o2n[t][k - plo_o]; kn = m < 0 ? -1 : plo_n + m; }
                cmap[k] = kn;
                if (kn >= 0) is_added[kn] = 0;
            }
            for (int k = ntsv_o; k < q_o; ++k) cmap[k] = ntsv_n + (k - ntsv_o);  // terminals keep their order
            std::vector<int> added;
            for (int k = 0; k < ntsv_n; ++k) if (is_added[k]) added.push_back(k);
            DevBuf d_cmap, d_added, d_isadd;
            d_cmap.alloc((size_t)q_o * sizeof(int));
            CK(cudaMemcpyAsync(d_cmap.p, cmap.data(), (size_t)q_o * sizeof(int), cudaMemcpyHostToDevice, L.s));
            N.ZT.alloc((size_t)rows_n * q_n * sizeof(double));
            CK(cudaMemsetAsync(N.ZT.p, 0, (size_t)rows_n * q_n * sizeof(double), L.s));
            L.run(KC_SMALL, 0, [&] { k_remap_zt<<<dim3(cdiv(q_o, 128), grid_rows(rows_o)), 128, 0, L.s>>>(T.ZT.as<double>(), rows_o, q_o, d_cmap.as<int>(), d_cmap.as<int>(), N.ZT.as<double>(), q_n); });
            N.zdiag.alloc((size_t)std::max(N.nterm, 1) * sizeof(double));  // the terminals' diagonal does not depend on the TSV plan
            if (N.nterm > 0) CK(cudaMemcpyAsync(N.zdiag.p, T.zdiag.p, (size_t)N.nterm * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
            N.d_node.alloc((size_t)q_n * sizeof(int));
            CK(cudaMemcpyAsync(N.d_node.p, N.node.data(), (size_t)q_n * sizeof(int), cudaMemcpyHostToDevice, L.s));
            CK(cudaStreamSynchronize(L.s));  // cmap / node (host vectors) were read
            if (!added.empty()) {
                if (!h_ready) { H.allocate(n); h_ready = true; }
                status = H.build(L, T.gx0.as<double>(), T.gy0.as<double>(), false, true);
                if (status != PDN_OK) break;
                const int Bmax = pick_batch(H, (int)added.size(), c->opts);
                Work W;
                if (H.nlev > 1) W.allocate(H, Bmax, q_n);
                status = reduce_tier(c, L, H, W, Bmax, N, added, {}, tabs);
                if (status != PDN_OK) { g_last_error = std::string("tier ") + std::to_string(t) + ": " + pdn_strerror(status); break; }
                new_solves += (int64_t)added.size();
                d_added.alloc(added.size() * sizeof(int));
                d_isadd.alloc((size_t)rows_n);
                CK(cudaMemcpyAsync(d_added.p, added.data(), added.size() * sizeof(int), cudaMemcpyHostToDevice, L.s));
                CK(cudaMemcpyAsync(d_isadd.p, is_added.data(), (size_t)rows_n, cudaMemcpyHostToDevice, L.s));
                L.run(KC_SMALL, 0, [&] { k_mirror_added<<<dim3(cdiv(added.size(), 128), grid_rows(rows_n)), 128, 0, L.s>>>(N.ZT.as<double>(), rows_n, q_n, d_added.as<int>(), (int)added.size(), d_isadd.as<unsigned char>()); });
                CK(cudaStreamSynchronize(L.s));
            }
        }
        CK(cudaEventRecord(ev[1], L.s));
        if (status == PDN_OK) {
            // ---- commit: from here on the context describes the new plan
            committed = true;
            for (int t = 0; t < d; ++t) {
                if (!changed[t]) continue;
                TierPorts& T = c->tiers[t];
                TierPorts& N = staged[t];
                T.node = std::move(N.node); T.ntsv = N.ntsv; T.nterm = N.nterm; T.q = N.q; T.nrows = N.nrows;
                T.d_node = std::move(N.d_node); T.ZT = std::move(N.ZT); T.zdiag = std::move(N.zdiag);
            }
            c->site = nsite;
            c->rt = nrt;
            c->stats.n_ports_total = 0;
            for (int i = 0; i < d - 1; ++i) c->p[i] = (int)nsite[i].size();
            for (int t = 0; t < d; ++t) c->stats.n_ports_total += c->tiers[t].q;
            status = recombine(c, L);
            if (status != PDN_OK) {  // the old factor is gone and the new one is incomplete: nothing but pdn_destroy is left
                g_last_error = std::string(pdn_strerror(status)) + " (the context is no longer usable: destroy it)";
                c->poisoned = true;
            }
        }
        CK(cudaEventRecord(ev[2], L.s));
        CK(cudaStreamSynchronize(L.s));
        L.resolve();
        float ms_s1 = 0.f, ms_dense = 0.f;
        CK(cudaEventElapsedTime(&ms_s1, ev[0], ev[1]));
        CK(cudaEventElapsedTime(&ms_dense, ev[1], ev[2]));
        c->stats.ms_update_stencil = ms_s1; c->stats.ms_update_dense = ms_dense; c->stats.update_solves = new_solves;
        for (auto& e : ev) cudaEventDestroy(e);
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        status = f.e == cudaErrorMemoryAllocation ? PDN_E_NOMEM : PDN_E_CUDA;
    } catch (const StatusFail& f) {
        g_last_error = f.msg;
        status = f.status;
    } catch (const std::bad_alloc&) {
        g_last_error = "host allocation failed";
        status = PDN_E_NOMEM;
    }
    if (status != PDN_OK && committed) c->poisoned = true;
    return status;
}

int pdn_set_solver_opts(pdn_ctx* ctx, double rtol, int32_t max_iter) {
    if (!ctx) return fail_arg("null context");
    if (rtol > 0.0) {
        if (!std::isfinite(rtol) || rtol >= 1.0) return fail_arg("rtol must be in (0, 1)");
        ctx->opts.rtol = rtol;
    }
    if (max_iter > 0) ctx->opts.max_iter = max_iter;
    return PDN_OK;
}

static int reff_device(pdn_ctx* ctx, int64_t n_pairs, const int32_t* bi, const int32_t* li, double* out) {
    Launcher L{ctx, ctx->stream};
    const int m = ctx->m, n = ctx->nl, p0 = ctx->p0;
    if (!bi) {
        dim3 grid(cdiv(n, 64), cdiv(m, 64));
        L.run(KC_PAIR, (double)n_pairs * 8.0, [&] { k_pair_full<<<grid, 256, 0, L.s>>>(m, n, p0, ctx->A1.as<double>(), ctx->X0.as<double>(), ctx->u.as<double>(), ctx->w.as<double>(), out); });
    } else {
        L.run(KC_PAIR, (double)n_pairs * 8.0, [&] { k_pair_list<<<cdiv((size_t)n_pairs * 32, 256), 256, 0, L.s>>>(n_pairs, m, n, p0, bi, li, ctx->A1.as<double>(), ctx->X0.as<double>(), ctx->u.as<double>(), ctx->w.as<double>(), out); });
    }
    return PDN_OK;
}

int pdn_reff(pdn_ctx* ctx, int64_t n_pairs, const int32_t* bump_idx, const int32_t* load_idx, double* out) {
    if (!ctx || !out || n_pairs < 0) return fail_arg("null context / output or negative n_pairs");
    PDN_CHECK_DEVICE(ctx);
    if (ctx->open) return fail_arg("sharded context is still open: exchange the rows and call pdn_finish first");
    if ((bump_idx == nullptr) != (load_idx == nullptr)) return fail_arg("bump_idx and load_idx must both be given or both be NULL");
    if (!bump_idx && n_pairs != (int64_t)ctx->m * ctx->nl) return fail_arg("full cross product needs n_pairs == n_bumps*n_loads");
    if (n_pairs == 0) return PDN_OK;
    try {
        reff_device(ctx, n_pairs, bump_idx, load_idx, out);
        CK(cudaStreamSynchronize(ctx->stream));
        Launcher{ctx, ctx->stream}.resolve();
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        return PDN_E_CUDA;
    }
    return PDN_OK;
}

int pdn_reff_host(pdn_ctx* ctx, int64_t n_pairs, const int32_t* bump_idx, const int32_t* load_idx, double* out) {
    if (!ctx || !out || n_pairs < 0) return fail_arg("null context / output or negative n_pairs");
    PDN_CHECK_DEVICE(ctx);
    if (ctx->open) return fail_arg("sharded context is still open: exchange the rows and call pdn_finish first");
    if ((bump_idx == nullptr) != (load_idx == nullptr)) return fail_arg("bump_idx and load_idx must both be given or both be NULL");
    if (!bump_idx && n_pairs != (int64_t)ctx->m * ctx->nl) return fail_arg("full cross product needs n_pairs == n_bumps*n_loads");
    if (n_pairs == 0) return PDN_OK;
    try {
        DevBuf dout, dbi, dli;
        dout.alloc((size_t)n_pairs * sizeof(double));
        if (bump_idx) {
            dbi.alloc((size_t)n_pairs * sizeof(int32_t));
            dli.alloc((size_t)n_pairs * sizeof(int32_t));
            CK(cudaMemcpyAsync(dbi.p, bump_idx, (size_t)n_pairs * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream));
            CK(cudaMemcpyAsync(dli.p, load_idx, (size_t)n_pairs * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream));
        }
        reff_device(ctx, n_pairs, bump_idx ? dbi.as<int32_t>() : nullptr, bump_idx ? dli.as<int32_t>() : nullptr, dout.as<double>());
        CK(cudaMemcpyAsync(out, dout.p, (size_t)n_pairs * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
        Launcher{ctx, ctx->stream}.resolve();
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        return PDN_E_CUDA;
    } catch (const StatusFail& f) {
        g_last_error = f.msg;
        return f.status;
    }
    return PDN_OK;
}

void pdn_release_cache(void) { g_pool.trim(); }

// NEXT-3: R_eff between terminals of the same side (bump-bump or load-load), full nt x nt matrix on the device.
int pdn_reff_same_side(pdn_ctx* ctx, int32_t side, double* out) {
    if (!ctx || !out || (side != 0 && side != 1)) return fail_arg("null context / output or side not in {0, 1}");
    PDN_CHECK_DEVICE(ctx);
    if (!ctx->terminal_pairs) return fail_arg("the context was not created with PDN_TERMINAL_PAIRS");
    if (ctx->open) return fail_arg("sharded context is still open: exchange the rows and call pdn_finish first");
    if (ctx->d < 2) return fail_arg("same-side pairs need at least 2 tiers (on one tier list the nodes as bumps and loads)");
    try {
        Launcher L{ctx, ctx->stream};
        const pdn_ctx::Side& S = ctx->side[side];
        const TierPorts& T = ctx->tiers[side == 0 ? 0 : ctx->d - 1];
        const int nt = T.nterm;
        dim3 grid(cdiv(nt, 64), cdiv(nt, 64));
        L.run(KC_PAIR, (double)nt * nt * 8.0, [&] { k_pair_same<<<grid, 256, 0, L.s>>>(nt, S.p, S.A.as<double>(), S.X.as<double>(), S.ys.as<double>(), S.t.as<double>(), T.ZT.as<double>(), T.q, T.ntsv, out); });
        CK(cudaStreamSynchronize(ctx->stream));
        L.resolve();
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        return PDN_E_CUDA;
    }
    return PDN_OK;
}

// NEXT-3: Eq. (4).
int pdn_load_voltages(pdn_ctx* ctx, int32_t bump, const double* i_load, double v_bump, double* v_out) {
    if (!ctx || !i_load || !v_out) return fail_arg("null argument");
    PDN_CHECK_DEVICE(ctx);
    if (!ctx->terminal_pairs) return fail_arg("the context was not created with PDN_TERMINAL_PAIRS");
    if (ctx->open) return fail_arg("sharded context is still open: exchange the rows and call pdn_finish first");
    if (bump < 0 || bump >= ctx->m) return fail_arg("bump index out of range");
    if (ctx->d < 2) return fail_arg("pdn_load_voltages needs at least 2 tiers");
    try {
        Launcher L{ctx, ctx->stream};
        const int n = ctx->nl, m = ctx->m, p0 = ctx->p0;
        DevBuf Rb, RLL, bi, li;
        Rb.alloc((size_t)n * sizeof(double));
        RLL.alloc((size_t)n * n * sizeof(double));
        bi.alloc((size_t)n * sizeof(int));
        li.alloc((size_t)n * sizeof(int));
        std::vector<int> hb(n, bump), hl(n);
        for (int k = 0; k < n; ++k) hl[k] = k;
        CK(cudaMemcpyAsync(bi.p, hb.data(), (size_t)n * sizeof(int), cudaMemcpyHostToDevice, L.s));
        CK(cudaMemcpyAsync(li.p, hl.data(), (size_t)n * sizeof(int), cudaMemcpyHostToDevice, L.s));
        // R_b[k] = R_eff(bump, load k): one row of the bump x load matrix
        L.run(KC_PAIR, (double)n * 8.0, [&] { k_pair_list<<<cdiv((size_t)n * 32, 256), 256, 0, L.s>>>(n, m, n, p0, bi.as<int>(), li.as<int>(), ctx->A1.as<double>(), ctx->X0.as<double>(), ctx->u.as<double>(), ctx->w.as<double>(), Rb.as<double>()); });
        const pdn_ctx::Side& S = ctx->side[1];
        const TierPorts& T = ctx->tiers[ctx->d - 1];
        dim3 grid(cdiv(n, 64), cdiv(n, 64));
        L.run(KC_PAIR, (double)n * n * 8.0, [&] { k_pair_same<<<grid, 256, 0, L.s>>>(n, S.p, S.A.as<double>(), S.X.as<double>(), S.ys.as<double>(), S.t.as<double>(), T.ZT.as<double>(), T.q, T.ntsv, RLL.as<double>()); });
        L.run(KC_PAIR, (double)n * n * 8.0, [&] { k_load_voltages<<<cdiv((size_t)n * 32, 256), 256, 0, L.s>>>(n, Rb.as<double>(), RLL.as<double>(), i_load, v_bump, v_out); });
        CK(cudaStreamSynchronize(ctx->stream));
        L.resolve();
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        return PDN_E_CUDA;
    } catch (const StatusFail& f) {
        g_last_error = f.msg;
        return f.status;
    }
    return PDN_OK;
}

// Eq. (4) with the scratch in g_static_scratch: no device pool, no cudaMalloc / cudaFree, no events, no host
// containers.  Three launches on the context's stream: k_pair_row (R_b), k_pair_same (R_LL), k_load_voltages.
int pdn_load_voltages_static(pdn_ctx* ctx, int32_t bump, const double* i_load, double v_bump, double* v_out) {
    if (!ctx || !i_load || !v_out) return fail_arg("null argument");
    PDN_CHECK_DEVICE(ctx);
    if (!ctx->terminal_pairs) return fail_arg("the context was not created with PDN_TERMINAL_PAIRS");
    if (ctx->open) return fail_arg("sharded context is still open: exchange the rows and call pdn_finish first");
    if (bump < 0 || bump >= ctx->m) return fail_arg("bump index out of range");
    if (ctx->d < 2) return fail_arg("pdn_load_voltages_static needs at least 2 tiers");
    if (ctx->nl > STATIC_MAXL)
        return fail_arg("pdn_load_voltages_static: n_loads exceeds PDN_STATIC_MAX_LOADS (512), the size of the library's "
                        "static scratch array; use pdn_load_voltages");
    try {
        double* scratch = static_scratch_of_current_device();
        const int n = ctx->nl, m = ctx->m, p0 = ctx->p0;
        double* RLL = scratch;
        double* Rb = scratch + (size_t)STATIC_MAXL * STATIC_MAXL;
        cudaStream_t s = ctx->stream;
        const pdn_ctx::Side& S = ctx->side[1];
        const TierPorts& T = ctx->tiers[ctx->d - 1];
        k_pair_row<<<cdiv((size_t)n * 32, 256), 256, 0, s>>>(bump, n, p0, ctx->A1.as<double>(), ctx->X0.as<double>(), ctx->u.as<double>(), ctx->w.as<double>(), Rb);
        CK(cudaGetLastError());
        dim3 grid(cdiv(n, 64), cdiv(n, 64));
        k_pair_same<<<grid, 256, 0, s>>>(n, S.p, S.A.as<double>(), S.X.as<double>(), S.ys.as<double>(), S.t.as<double>(), T.ZT.as<double>(), T.q, T.ntsv, RLL);
        CK(cudaGetLastError());
        k_load_voltages<<<cdiv((size_t)n * 32, 256), 256, 0, s>>>(n, Rb, RLL, i_load, v_bump, v_out);
        CK(cudaGetLastError());
        {
            std::lock_guard<std::mutex> g(ctx->mu);
            ctx->class_launches[KC_PAIR] += 3;
            ctx->class_bytes[KC_PAIR] += (2.0 * n * n + n) * 8.0;
            ctx->stats.kernel_launches += 3;
        }
        // complete on return like every other entry point -- unless the stream is being captured into a CUDA graph,
        // where a synchronise would end the capture: then the three kernel nodes are all the call leaves behind
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        CK(cudaStreamIsCapturing(s, &cap));
        if (cap == cudaStreamCaptureStatusNone) CK(cudaStreamSynchronize(s));
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        return PDN_E_CUDA;
    } catch (const StatusFail& f) {
        g_last_error = f.msg;
        return f.status;
    }
    return PDN_OK;
}

// NEXT-3: arbitrary-tier endpoints (port.cuh "Arbitrary-tier endpoints" has the algebra).
int pdn_reff_nodes(pdn_ctx* ctx, int32_t n_nodes, const pdn_node* nodes, double* out) {
    if (!ctx || !nodes || !out || n_nodes < 1) return fail_arg("null context / node list / output or empty list");
    PDN_CHECK_DEVICE(ctx);
    if (ctx->open) return fail_arg("sharded context is still open: exchange the rows and call pdn_finish first");
    if (ctx->d < 2) return fail_arg("pdn_reff_nodes needs at least 2 tiers (on one tier list the nodes as bumps and loads)");
    pdn_ctx* c = ctx;
    const int d = c->d, n = c->n, dm1 = d - 1, np = n_nodes;
    for (int a = 0; a < np; ++a) {
        if (nodes[a].tier < 0 || nodes[a].tier >= d) return fail_arg("probe tier out of range");
        if (nodes[a].y < 0 || nodes[a].y >= n || nodes[a].x < 0 || nodes[a].x >= n) return fail_arg("probe site out of range");
    }
    int status = PDN_OK;
    const pdn_stats stats0 = c->stats;  // the solve statistics describe pdn_create / pdn_update_tsvs only
    try {
        Launcher L{c, c->stream};
        std::vector<DevBuf> F(dm1), X(dm1);
        DevBuf M, G, Cs, mu, d_tier;
        for (int i = 0; i < dm1; ++i) {
            F[i].alloc((size_t)c->p[i] * np * sizeof(double));
            X[i].alloc((size_t)c->p[i] * np * sizeof(double));
            CK(cudaMemsetAsync(F[i].p, 0, (size_t)c->p[i] * np * sizeof(double), L.s));
        }
        M.alloc((size_t)np * np * sizeof(double));
        CK(cudaMemsetAsync(M.p, 0, (size_t)np * np * sizeof(double), L.s));
        std::vector<int> h_tier(np);
        for (int a = 0; a < np; ++a) h_tier[a] = nodes[a].tier;
        d_tier.alloc((size_t)np * sizeof(int));
        CK(cudaMemcpyAsync(d_tier.p, h_tier.data(), (size_t)np * sizeof(int), cudaMemcpyHostToDevice, L.s));
        // ---- one port solve per probe, tier by tier
        SpectralTables tabs;
        Hierarchy H;
        bool h_ready = false;
        for (int t = 0; t < d && status == PDN_OK; ++t) {
            std::vector<int> probe;
            for (int a = 0; a < np; ++a) if (nodes[a].tier == t) probe.push_back(a);
            if (probe.empty()) continue;
            const TierPorts& T = c->tiers[t];
            const int k = (int)probe.size();
            TierPorts Tp;
            Tp.node.assign(T.node.begin(), T.node.begin() + T.ntsv);
            for (int a : probe) Tp.node.push_back(nodes[a].y * pitch_of(n) + nodes[a].x);
            Tp.ntsv = T.ntsv; Tp.nterm = k; Tp.q = T.ntsv + k; Tp.nrows = Tp.q;
            Tp.d_node.alloc((size_t)Tp.q * sizeof(int));
            CK(cudaMemcpyAsync(Tp.d_node.p, Tp.node.data(), (size_t)Tp.q * sizeof(int), cudaMemcpyHostToDevice, L.s));
            Tp.ZT.alloc((size_t)Tp.q * Tp.q * sizeof(double));
            Tp.zdiag.alloc((size_t)k * sizeof(double));
            if (!h_ready) { H.allocate(n); h_ready = true; }
            status = H.build(L, T.gx0.as<double>(), T.gy0.as<double>(), false, true);
            if (status != PDN_OK) break;
            const int Bmax = pick_batch(H, k, c->opts);
            Work W;
            if (H.nlev > 1) W.allocate(H, Bmax, Tp.q);
            std::vector<int> src(k);
            for (int j = 0; j < k; ++j) src[j] = T.ntsv + j;
            status = reduce_tier(c, L, H, W, Bmax, Tp, src, {}, tabs);
            if (status != PDN_OK) { g_last_error = std::string("tier ") + std::to_string(t) + ": " + pdn_strerror(status); break; }
            DevBuf d_probe;
            d_probe.alloc((size_t)k * sizeof(int));
            CK(cudaMemcpyAsync(d_probe.p, probe.data(), (size_t)k * sizeof(int), cudaMemcpyHostToDevice, L.s));
            const int plo = t > 0 ? c->p[t - 1] : 0;
            double* Fup = t < dm1 ? F[t].as<double>() : nullptr;
            double* Flo = t > 0 ? F[t - 1].as<double>() : nullptr;
            L.run(KC_DENSE, 0, [&] { k_probe_scatter<<<dim3(cdiv(Tp.q, 128), grid_rows(k)), 128, 0, L.s>>>(k, T.ntsv, plo, np, d_probe.as<int>(), Tp.ZT.as<double>(), Fup, Flo, M.as<double>()); });
            CK(cudaStreamSynchronize(L.s));  // probe (host vector) and the tier's buffers are released here
        }
        if (status == PDN_OK) {
            // ---- X = currents of C^-1 [F; Cs];  M -= F^T X + Cs^T mu
            for (int i = 0; i < dm1; ++i) CK(cudaMemcpyAsync(X[i].p, F[i].p, (size_t)c->p[i] * np * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
            block_substitute(c, L, X, np);
            G.alloc((size_t)dm1 * np * sizeof(double));
            Cs.alloc((size_t)dm1 * np * sizeof(double));
            mu.alloc((size_t)dm1 * np * sizeof(double));
            for (int i = 0; i < dm1; ++i)
                L.run(KC_DENSE, 0, [&] { k_colsum<<<cdiv(np, 128), 128, 0, L.s>>>(c->p[i], np, X[i].as<double>(), G.as<double>() + (size_t)i * np); });
            L.run(KC_DENSE, 0, [&] { k_probe_multipliers<<<cdiv(np, 128), 128, 0, L.s>>>(dm1, np, G.as<double>(), c->Sinv.as<double>(), d_tier.as<int>(), Cs.as<double>(), mu.as<double>()); });
            for (int i = 0; i < dm1; ++i) {
                const int pi = c->p[i];
                gemm(L, pi, np, dm1, -1.0, c->KB[i].as<double>(), dm1, 1, mu.as<double>(), np, 1, 1.0, X[i].as<double>(), np);
                gemm(L, np, np, pi, -1.0, F[i].as<double>(), 1, np, X[i].as<double>(), np, 1, 1.0, M.as<double>(), np);
            }
            gemm(L, np, np, dm1, -1.0, Cs.as<double>(), 1, np, mu.as<double>(), np, 1, 1.0, M.as<double>(), np);
            L.run(KC_PAIR, (double)np * np * 8.0, [&] { k_probe_pairs<<<dim3(cdiv(np, 128), grid_rows(np)), 128, 0, L.s>>>(np, M.as<double>(), out); });
        }
        CK(cudaStreamSynchronize(L.s));
        L.resolve();
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        status = f.e == cudaErrorMemoryAllocation ? PDN_E_NOMEM : PDN_E_CUDA;
    } catch (const StatusFail& f) {
        g_last_error = f.msg;
        status = f.status;
    } catch (const std::bad_alloc&) {
        g_last_error = "host allocation failed";
        status = PDN_E_NOMEM;
    }
    const int64_t launches = c->stats.kernel_launches, stencil_launches = c->stats.stencil_launches;
    c->stats = stats0;
    c->stats.kernel_launches = launches;
    c->stats.stencil_launches = stencil_launches;
    return status;
}

// NEXT-3: one source against many nodes (port.cuh: k_from_scatter has the algebra).
int pdn_reff_from(pdn_ctx* ctx, const pdn_node* src_node, int32_t n_nodes, const pdn_node* nodes, double* out) {
    if (!ctx || !src_node || !nodes || !out || n_nodes < 1) return fail_arg("null context / source / node list / output or empty list");
    PDN_CHECK_DEVICE(ctx);
    if (ctx->open) return fail_arg("sharded context is still open: exchange the rows and call pdn_finish first");
    if (ctx->d < 2) return fail_arg("pdn_reff_from needs at least 2 tiers (on one tier list the nodes as bumps and loads)");
    pdn_ctx* c = ctx;
    const int d = c->d, n = c->n, dm1 = d - 1, np = n_nodes + 1;
    std::vector<pdn_node> pr(np);
    pr[0] = *src_node;
    for (int a = 1; a < np; ++a) pr[a] = nodes[a - 1];
    for (int a = 0; a < np; ++a) {
        if (pr[a].tier < 0 || pr[a].tier >= d) return fail_arg("probe tier out of range");
        if (pr[a].y < 0 || pr[a].y >= n || pr[a].x < 0 || pr[a].x >= n) return fail_arg("probe site out of range");
    }
    int status = PDN_OK;
    const pdn_stats stats0 = c->stats;  // the solve statistics describe pdn_create / pdn_update_tsvs only
    try {
        Launcher L{c, c->stream};
        std::vector<DevBuf> F(dm1), X(dm1);
        DevBuf Zd, Zs, qd, qs, G, Cs, mu, d_tier;
        for (int i = 0; i < dm1; ++i) {
            F[i].alloc((size_t)c->p[i] * np * sizeof(double));
            X[i].alloc((size_t)c->p[i] * np * sizeof(double));
            CK(cudaMemsetAsync(F[i].p, 0, (size_t)c->p[i] * np * sizeof(double), L.s));
        }
        Zd.alloc((size_t)np * sizeof(double)); Zs.alloc((size_t)np * sizeof(double));
        qd.alloc((size_t)np * sizeof(double)); qs.alloc((size_t)np * sizeof(double));
        for (DevBuf* b : {&Zd, &Zs, &qd, &qs}) CK(cudaMemsetAsync(b->p, 0, (size_t)np * sizeof(double), L.s));
        std::vector<int> h_tier(np);
        for (int a = 0; a < np; ++a) h_tier[a] = pr[a].tier;
        d_tier.alloc((size_t)np * sizeof(int));
        CK(cudaMemcpyAsync(d_tier.p, h_tier.data(), (size_t)np * sizeof(int), cudaMemcpyHostToDevice, L.s));
        // ---- per tier with probes: TSV-port solves gathered at the probes (+ the source's own row), one diagonal solve per probe
        SpectralTables tabs;
        Hierarchy H;
        bool h_ready = false;
        for (int t = 0; t < d && status == PDN_OK; ++t) {
            std::vector<int> probe;  // columns of the np-wide arrays; the source first if it sits on this tier
            for (int a = 0; a < np; ++a) if (pr[a].tier == t) probe.push_back(a);
            if (probe.empty()) continue;
            const TierPorts& T = c->tiers[t];
            const bool has_src = pr[0].tier == t;
            const int k = (int)probe.size(), nrow = T.ntsv + (has_src ? 1 : 0), kterm = k - (has_src ? 1 : 0);
            TierPorts Tp;
            Tp.node.assign(T.node.begin(), T.node.begin() + T.ntsv);
            for (int a : probe) Tp.node.push_back(pr[a].y * pitch_of(n) + pr[a].x);
            Tp.ntsv = nrow; Tp.nterm = kterm; Tp.q = T.ntsv + k; Tp.nrows = nrow;
            Tp.d_node.alloc((size_t)Tp.q * sizeof(int));
            CK(cudaMemcpyAsync(Tp.d_node.p, Tp.node.data(), (size_t)Tp.q * sizeof(int), cudaMemcpyHostToDevice, L.s));
            Tp.ZT.alloc((size_t)std::max(nrow, 1) * Tp.q * sizeof(double));
            Tp.zdiag.alloc((size_t)std::max(kterm, 1) * sizeof(double));
            if (!h_ready) { H.allocate(n); h_ready = true; }
            status = H.build(L, T.gx0.as<double>(), T.gy0.as<double>(), false, true);
            if (status != PDN_OK) break;
            const int Bmax = pick_batch(H, Tp.q, c->opts);
            Work W;
            if (H.nlev > 1) W.allocate(H, Bmax, Tp.q);
            std::vector<int> rows(nrow), term(kterm);
            for (int j = 0; j < nrow; ++j) rows[j] = j;
            for (int j = 0; j < kterm; ++j) term[j] = nrow + j;
            status = reduce_tier(c, L, H, W, Bmax, Tp, rows, term, tabs, true);
            if (status != PDN_OK) { g_last_error = std::string("tier ") + std::to_string(t) + ": " + pdn_strerror(status); break; }
            std::vector<int> col(k);
            for (int j = 0; j < k; ++j) col[j] = T.ntsv + j;
            DevBuf d_probe, d_col;
            d_probe.alloc((size_t)k * sizeof(int)); d_col.alloc((size_t)k * sizeof(int));
            CK(cudaMemcpyAsync(d_probe.p, probe.data(), (size_t)k * sizeof(int), cudaMemcpyHostToDevice, L.s));
            CK(cudaMemcpyAsync(d_col.p, col.data(), (size_t)k * sizeof(int), cudaMemcpyHostToDevice, L.s));
            const int plo = t > 0 ? c->p[t - 1] : 0;
            double* Fup = t < dm1 ? F[t].as<double>() : nullptr;
            double* Flo = t > 0 ? F[t - 1].as<double>() : nullptr;
            L.run(KC_DENSE, 0, [&] { k_from_scatter<<<dim3(cdiv((size_t)T.ntsv + 1, 128), grid_rows(k)), 128, 0, L.s>>>(k, T.ntsv, nrow, plo, np, has_src ? T.ntsv : -1, d_col.as<int>(), d_probe.as<int>(), Tp.ZT.as<double>(), Tp.q, Tp.zdiag.as<double>(), Fup, Flo, Zd.as<double>(), Zs.as<double>()); });
            CK(cudaStreamSynchronize(L.s));  // the host vectors and the tier's buffers are released here
        }
        if (status == PDN_OK) {
            // ---- X = currents of C^-1 [F; Cs] for all np columns; then one row and the diagonal of M
            for (int i = 0; i < dm1; ++i) CK(cudaMemcpyAsync(X[i].p, F[i].p, (size_t)c->p[i] * np * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
            block_substitute(c, L, X, np);
            G.alloc((size_t)dm1 * np * sizeof(double));
            Cs.alloc((size_t)dm1 * np * sizeof(double));
            mu.alloc((size_t)dm1 * np * sizeof(double));
            for (int i = 0; i < dm1; ++i)
                L.run(KC_DENSE, 0, [&] { k_colsum<<<cdiv(np, 128), 128, 0, L.s>>>(c->p[i], np, X[i].as<double>(), G.as<double>() + (size_t)i * np); });
            L.run(KC_DENSE, 0, [&] { k_probe_multipliers<<<cdiv(np, 128), 128, 0, L.s>>>(dm1, np, G.as<double>(), c->Sinv.as<double>(), d_tier.as<int>(), Cs.as<double>(), mu.as<double>()); });
            for (int i = 0; i < dm1; ++i) {
                const int pi = c->p[i];
                gemm(L, pi, np, dm1, -1.0, c->KB[i].as<double>(), dm1, 1, mu.as<double>(), np, 1, 1.0, X[i].as<double>(), np);
                L.run(KC_DENSE, 0, [&] { k_from_dots<<<cdiv(np, 128), 128, 0, L.s>>>(pi, np, F[i].as<double>(), X[i].as<double>(), qd.as<double>(), qs.as<double>()); });
            }
            L.run(KC_PAIR, (double)np * 8.0, [&] { k_from_finish<<<cdiv(np, 128), 128, 0, L.s>>>(dm1, np, Cs.as<double>(), mu.as<double>(), Zd.as<double>(), Zs.as<double>(), qd.as<double>(), qs.as<double>(), out); });
        }
        CK(cudaStreamSynchronize(L.s));
        L.resolve();
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        status = f.e == cudaErrorMemoryAllocation ? PDN_E_NOMEM : PDN_E_CUDA;
    } catch (const StatusFail& f) {
        g_last_error = f.msg;
        status = f.status;
    } catch (const std::bad_alloc&) {
        g_last_error = "host allocation failed";
        status = PDN_E_NOMEM;
    }
    const int64_t launches = c->stats.kernel_launches, stencil_launches = c->stats.stencil_launches;
    c->stats = stats0;
    c->stats.kernel_launches = launches;
    c->stats.stencil_launches = stencil_launches;
    return status;
}

int pdn_shard_slice(const pdn_ctx* ctx, int32_t tier, int32_t rank, int32_t* tsv0, int32_t* ntsv, int32_t* term0,
                    int32_t* nterm) {
    if (!ctx || !tsv0 || !ntsv || !term0 || !nterm || tier < 0 || tier >= ctx->d || rank < 0 || rank >= ctx->shard_world)
        return fail_arg("bad tier / rank or null output");
    const TierPorts& T = ctx->tiers[tier];
    const int64_t W_ = ctx->shard_world;
    *tsv0 = *ntsv = *term0 = *nterm = 0;
    if (T.whole || W_ <= 1) return PDN_OK;
    *tsv0 = (int32_t)(rank * (int64_t)T.ntsv / W_);
    *ntsv = (int32_t)((rank + 1) * (int64_t)T.ntsv / W_) - *tsv0;
    *term0 = (int32_t)(rank * (int64_t)T.nterm / W_);
    *nterm = (int32_t)((rank + 1) * (int64_t)T.nterm / W_) - *term0;
    return PDN_OK;
}

int pdn_shard_buffers(pdn_ctx* ctx, int32_t tier, double** zt, int64_t* ld, int32_t* ntsv_total, double** zdiag) {
    if (!ctx || !zt || !ld || !ntsv_total || !zdiag || tier < 0 || tier >= ctx->d) return fail_arg("bad tier or null output");
    TierPorts& T = ctx->tiers[tier];
    *zt = T.ZT.as<double>(); *ld = T.q; *ntsv_total = T.ntsv; *zdiag = T.zdiag.as<double>();
    return PDN_OK;
}

int pdn_finish(pdn_ctx* ctx) {
    if (!ctx) return fail_arg("null context");
    PDN_CHECK_DEVICE(ctx);
    if (!ctx->open) return PDN_OK;
    int status = PDN_OK;
    try {
        Launcher L{ctx, ctx->stream};
        cudaEvent_t ev[2];
        for (auto& e : ev) CK(cudaEventCreate(&e));
        CK(cudaEventRecord(ev[0], L.s));
        if (ctx->terminal_pairs)
            for (TierPorts& T : ctx->tiers)
                if (T.nterm > 0 && !T.whole)
                    L.run(KC_SMALL, 0, [&] { k_zdiag_from_rows<<<cdiv(T.nterm, 128), 128, 0, L.s>>>(T.ZT.as<double>(), T.q, T.ntsv, T.nterm, T.zdiag.as<double>()); });
        status = recombine(ctx, L);
        if (status != PDN_OK) g_last_error = pdn_strerror(status);
        CK(cudaEventRecord(ev[1], L.s));
        CK(cudaStreamSynchronize(L.s));
        L.resolve();
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, ev[0], ev[1]));
        ctx->stats.ms_dense = ms;
        ctx->stats.ms_total += ms;
        for (auto& e : ev) cudaEventDestroy(e);
        if (status == PDN_OK) ctx->open = false;
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        cudaGetLastError();
        status = f.e == cudaErrorMemoryAllocation ? PDN_E_NOMEM : PDN_E_CUDA;
    } catch (const StatusFail& f) {
        g_last_error = f.msg;
        status = f.status;
    }
    return status;
}

int pdn_get_stats(const pdn_ctx* ctx, pdn_stats* out) {
    if (!ctx || !out) return fail_arg("null argument");
    *out = ctx->stats;
    out->stencil_bytes = 0.0;
    for (int k = 0; k < KC_COUNT; ++k) {
        out->class_ms[k] = ctx->class_ms[k];
        out->class_bytes[k] = ctx->class_bytes[k];
        out->class_launches[k] = ctx->class_launches[k];
        if (k <= KC_SMALL) out->stencil_bytes += ctx->class_bytes[k];
    }
    return PDN_OK;
}

int32_t pdn_port_count(const pdn_ctx* ctx, int32_t tier) {
    if (!ctx || tier < 0 || tier >= ctx->d) return -1;
    return ctx->tiers[tier].q;
}

int pdn_get_port_matrix(const pdn_ctx* ctx, int32_t tier, double* out) {
    if (!ctx || !out || tier < 0 || tier >= ctx->d) return fail_arg("bad tier or null output");
    if (ctx->poisoned) return fail_arg("the context is unusable after a failed pdn_update_tsvs: destroy it");
    const TierPorts& T = ctx->tiers[tier];
    try {
        std::vector<double> zt((size_t)T.nrows * T.q), zd((size_t)T.nterm);
        CK(cudaMemcpy(zt.data(), T.ZT.p, zt.size() * sizeof(double), cudaMemcpyDeviceToHost));
        if (T.nterm) CK(cudaMemcpy(zd.data(), T.zdiag.p, zd.size() * sizeof(double), cudaMemcpyDeviceToHost));
        const double qnan = std::nan("");
        for (int j = 0; j < T.q; ++j)
            for (int k = 0; k < T.q; ++k) {
                double v = qnan;
                if (j < T.nrows && k < T.nrows) v = 0.5 * (zt[(size_t)j * T.q + k] + zt[(size_t)k * T.q + j]);
                else if (j < T.nrows) v = zt[(size_t)j * T.q + k];
                else if (k < T.nrows) v = zt[(size_t)k * T.q + j];
                else if (j == k) v = zd[j - T.ntsv];
                out[(size_t)j * T.q + k] = v;
            }
    } catch (const CudaFail& f) {
        g_last_error = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        return PDN_E_CUDA;
    }
    return PDN_OK;
}

}  // extern "C"
