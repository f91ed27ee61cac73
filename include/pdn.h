/*
 * pdn.h -- C ABI of the B200-native bump x load effective-resistance path.
 *
 * What the library computes: for a 3D-IC power delivery network modelled as a resistor network
 * (d stacked 2D meshes joined by TSVs), the effective resistance
 *
 *      R_eff(b, l) = (e_b - e_l)^T G^+ (e_b - e_l)                  PAPER.md:40-43, Eq. (2)
 *
 * between bump b (a node of the top tier) and load l (a node of the bottom tier), for every
 * requested pair, by the paper's divide-and-conquer method:
 *   S1  each tier is reduced to its port nodes (TSV sites, bumps, loads) by batched
 *       multi-right-hand-side solves on its 2D 5-point stencil (intra-die effective resistances,
 *       the d x p x p, m x p, n x p arrays),
 *   S2  the reusable coefficient matrix C = [K B; B^T 0] of Eq. (18) is assembled,
 *   S3  decomposed ONCE and solved for the m + n right-hand sides b^1_i, b^d_j of
 *       Eq. (21),
 *   S4  R_eff(i, j) = -(x^1_i + x^d_j)^T (b^1_i + b^d_j), Eq. (22), for all pairs.
 * pdn_create does S1-S3 (all the expensive work), pdn_reff does S4 and may be called repeatedly.
 *
 * Conventions.  0-based.  Tier 0 is the top tier (bumps; the paper's die_1), tier d-1 the bottom
 * tier (loads; die_d).  Tier t is an n x n node mesh, node (y, x), local id y*n + x.  Interface i
 * (0 <= i < d-1) joins tier i and tier i+1.  All arithmetic is IEEE FP64 (the diagonal scaling
 * inside the multigrid preconditioner uses FP32-representable factors, applied in FP64; the operator,
 * the residuals and every result are FP64).  A tier whose x-segments are all equal and whose
 * y-segments are all equal is reduced by the closed form, Eq. (3).  Every entry point
 * is thread-compatible (one thread per context at a time), never throws, and returns a status
 * (0 = PDN_OK).  A context lives on the CUDA device that is current when pdn_create is called; later
 * calls on it must be made with that device current (PDN_E_ARG otherwise).  A process may hold contexts
 * on several devices; freed device memory is cached per device (pdn_release_cache).  There is NO CPU
 * fallback: without a CUDA device every compute call fails with PDN_E_CUDA.
 */
#ifndef PDN_H_
#define PDN_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pdn_ctx pdn_ctx; /* opaque; owned by the library; freed by pdn_destroy */

/* status codes */
enum {
    PDN_OK = 0,
    PDN_E_ARG = 1,          /* null pointer, negative size, d < 2, n < 2, site / interface out of range,
                               r_ohm <= 0 or not finite, an interface without TSVs, a duplicate TSV site
                               inside one interface, negative / non-finite conductance                    */
    PDN_E_DISCONNECTED = 2, /* a tier is not one connected component (checked on the device)            */
    PDN_E_NOCONV = 3,       /* a port solve did not reach rtol within max_iter iterations               */
    PDN_E_CUDA = 4,         /* CUDA runtime error (pdn_last_error() has the string)                      */
    PDN_E_NOMEM = 5,        /* device or host allocation failed                                          */
    PDN_E_NUMERIC = 6       /* the port-level matrix K was not positive definite (should not happen for
                               a connected network with r_ohm > 0)                                        */
};

/* flags for pdn_opts.flags */
enum {
    PDN_TIERS_ON_HOST = 1,  /* pdn_tier.gx / gy are HOST pointers (the library uploads them)            */
    PDN_SKIP_CONNECTIVITY_CHECK = 2,
    PDN_TIME_KERNELS = 4,   /* bracket every kernel launch with CUDA events (per-class timers in pdn_stats) */
    PDN_TERMINAL_PAIRS = 16, /* also keep the bump-source / load-source rows of the port matrices (full tolerance,
                               gathered at every port): needed by pdn_reff_same_side and pdn_load_voltages; costs
                               about as much again as the bump / load part of pdn_create                        */
    PDN_PRECOND_F32 = 32,   /* opt-in mixed precision: the sweeps of the multigrid preconditioner (V-cycle stages
                               above the fused coarse tail) run in FP32 registers.  The CG operator, residuals,
                               step lengths, solutions, port matrices and everything after S1 stay FP64, every
                               vector in HBM stays FP64, and the solves still stop at the FP64 residual test, so
                               the results meet the same tolerance; only the iteration count may change.
                               Off by default: the default path computes in FP64 throughout                    */
    PDN_NO_INITIAL_GUESS = 64, /* start every port solve from x0 = 0 (default: on a mesh of n >= 192 whose segment
                               conductances scatter around their mean -- coefficient of variation <= 0.5 -- the
                               solves start from the closed form, Eq. (3), of the mean mesh; same stopping test,
                               same accuracy, about one PCG iteration less)                                      */
    PDN_NO_UNIFORM_FAST_PATH = 8 /* solve uniform tiers numerically too (default: a tier whose x-segments are all
                               equal and whose y-segments are all equal is reduced by the closed form, Eq. (3),
                               when it has enough ports for the 12 n^3-flop table to be cheaper than the solves) */
};

/* kernel classes of pdn_stats.class_* */
enum {
    PDN_KC_PQ = 0,     /* p = z + beta p ; q = L p ; p.q               (level 0)                   */
    PDN_KC_DOWN0 = 1,  /* r -= alpha q ; pre-smooth ; residual ; restrict (level 0)                 */
    PDN_KC_UP0 = 2,    /* prolong + correct ; post-smooth ; r.z          (level 0)                  */
    PDN_KC_DOWNC = 3,  /* down stages of the coarse levels                                          */
    PDN_KC_UPC = 4,    /* up stages of the coarse levels                                            */
    PDN_KC_SMALL = 5,  /* scalars, port gather, right-hand-side setup, hierarchy setup              */
    PDN_KC_DENSE = 6,  /* S2 + S3 port algebra                                                      */
    PDN_KC_PAIR = 7,   /* S4 pair evaluation                                                        */
    PDN_KC_COUNT = 8
};

/* One tier: an n x n mesh with per-edge conductances in siemens (0 = segment absent).
 *   gx[y*n + x] joins (y,x)-(y,x+1); the last column (x = n-1) is ignored.
 *   gy[y*n + x] joins (y,x)-(y+1,x); the last row    (y = n-1) is ignored.
 * gx, gy are DEVICE pointers (HOST pointers if PDN_TIERS_ON_HOST), n*n doubles each, row-major.
 * The library copies what it needs during pdn_create: the caller may free them afterwards. */
typedef struct {
    int32_t n;
    const double *gx;
    const double *gy;
} pdn_tier;

/* One TSV: joins node (y,x) of tier iface with node (y,x) of tier iface+1, resistance r_ohm
 * (Table I: Rt_k^{i,i+1}).  HOST array. */
typedef struct {
    int32_t iface, y, x;
    double r_ohm;
} pdn_tsv;

/* A bump (tier 0) or a load (tier d-1) node.  HOST arrays. */
typedef struct {
    int32_t y, x;
} pdn_site;

/* Options; pass NULL for the defaults.  Zero / negative fields mean "default". */
typedef struct {
    double rtol;        /* port solves stop at ||r||_2 <= rtol * ||b||_2          (default 1e-8);
                           bump / load sources, of which only the diagonal entry is used (its error is
                           quadratic in the residual), stop at min(1e-5, sqrt(rtol)/3, 1000 rtol)        */
    int32_t max_iter;   /* iteration cap per port solve                           (default 200)   */
    int32_t rhs_batch;  /* right-hand sides solved concurrently per tier          (default: auto) */
    void *cuda_stream;  /* cudaStream_t to run on                                 (default: 0)    */
    int32_t flags;      /* PDN_* flags                                                             */
    int32_t nu;         /* Chebyshev smoothing steps per multigrid level and side (1..6; default 4, and 6 on
                           tiers whose anisotropy mean g_x / mean g_y (or its inverse) is >= 6)             */
    double cheb_ratio;  /* smoothing interval [2/ratio, 2] of D^-1 L (default: 3 + the tier's anisotropy a,
                           2 (1 + a) for a >= 6)                                                             */
    int32_t shard_rank; /* NEXT-4: this process solves slice shard_rank of shard_world of every tier's port     */
    int32_t shard_world;/* solves and leaves the context OPEN (see pdn_shard_slice / pdn_finish); 0 or 1 = off  */
} pdn_opts;

/* Counters and timings of the last pdn_create (device-event milliseconds). */
typedef struct {
    int32_t n_tiers, n_ports_total, n_levels, n_uniform_tiers; /* tiers reduced by Eq. (3) */
    int64_t kernel_launches;     /* kernels launched by pdn_create so far (+ pdn_reff calls)      */
    int64_t stencil_launches;    /* of which S1 (stencil phase) kernels                            */
    int32_t pcg_iters_max;       /* max PCG iterations over all port-solve batches                */
    int32_t pcg_iters_sum;       /* sum over batches of the batch's iteration count               */
    int64_t rhs_iterations;      /* sum over iterations of the right-hand sides still iterating     */
    double worst_rel_residual;   /* max over all port solves of ||r|| / ||b|| at exit             */
    double ms_upload, ms_stencil, ms_dense, ms_total;
    double stencil_bytes;        /* algorithmic HBM bytes of the stencil phase (DESIGN.md model)  */
    double ms_update_stencil, ms_update_dense; /* last pdn_update_tsvs: port solves + remap / S2 + S3     */
    int64_t update_solves;       /* port solves the last pdn_update_tsvs needed                   */
    double class_ms[8];          /* device ms per kernel class (only with PDN_TIME_KERNELS)       */
    double class_bytes[8];       /* algorithmic bytes moved per kernel class                      */
    int64_t class_launches[8];   /* launches per kernel class                                     */
    int32_t n_guess_tiers;       /* tier reductions whose port solves started from the closed-form guess */
    int32_t n_guess_rejected;    /* right-hand sides of those whose guess did not help and that started from x0 = 0 */
} pdn_stats;

/* S0-S3.  tiers: HOST array of n_tiers descriptors (all tiers must have the same n).  tsvs, bumps,
 * loads: HOST arrays, copied.  On success *out owns all device memory it needs for pdn_reff.
 * Work is ordered on opts->cuda_stream; the call returns after that work completed.
 * n_tiers >= 2 needs at least one TSV on every interface.  n_tiers == 1 is the degenerate 2-D PDN (bumps and
 * loads on the one mesh, n_tsv == 0, tsvs may be NULL): R_eff is then Eq. (2) on that mesh, by the same port
 * solves and no recombination; pdn_update_tsvs, pdn_reff_same_side, pdn_load_voltages and pdn_reff_nodes need
 * n_tiers >= 2. */
int pdn_create(pdn_ctx **out, int32_t n_tiers, const pdn_tier *tiers,
               int32_t n_tsv, const pdn_tsv *tsvs,
               int32_t n_bumps, const pdn_site *bumps,
               int32_t n_loads, const pdn_site *loads,
               const pdn_opts *opts);

/* S4.  bump_idx / load_idx: DEVICE int32 arrays of length n_pairs indexing the create-time bump and
 * load lists; both NULL => the full cross product, out[i*n_loads + j], and n_pairs must equal
 * n_bumps*n_loads.  out: DEVICE fp64, caller-owned, n_pairs values; complete when the call returns.
 * An index out of range yields NaN in that slot (no error). */
int pdn_reff(pdn_ctx *ctx, int64_t n_pairs, const int32_t *bump_idx, const int32_t *load_idx, double *out);

/* Same with HOST index arrays (or NULL, NULL) and a HOST output buffer (S4 + S5: PAPER.md:218,
 * "transferred back to the CPU host"). */
int pdn_reff_host(pdn_ctx *ctx, int64_t n_pairs, const int32_t *bump_idx, const int32_t *load_idx, double *out);

/* TSV re-planning (the paper's design-space use case): replaces the TSV set of ctx by
 * the given list (HOST array, same rules as in pdn_create) and brings ctx up to date for pdn_reff.  The list is
 * diffed against the current one per interface by site: kept sites cost nothing (their resistance may change),
 * removed sites cost nothing, every added site costs one port solve on each of its two tiers; the port-level
 * system is then re-assembled and re-factored.  The update is staged: if a port solve fails (PDN_E_NOCONV,
 * PDN_E_NOMEM, PDN_E_CUDA, PDN_E_NUMERIC from a solve) or the list is malformed (PDN_E_ARG), ctx is left exactly as it
 * was and still answers for the OLD plan.  Only a failure of the final re-factorisation (PDN_E_NUMERIC from S3, or a
 * CUDA / allocation error inside it) leaves no valid factor: ctx is then marked unusable, every later call on it
 * returns PDN_E_ARG, and it must be destroyed. */
int pdn_update_tsvs(pdn_ctx *ctx, int32_t n_tsv, const pdn_tsv *tsvs);

/* Changes the stopping rule of the port solves that later calls on ctx run (pdn_update_tsvs, pdn_reff_nodes): the
 * relative residual rtol and the iteration cap max_iter of pdn_opts; a value <= 0 keeps the current one.  Design-
 * space sweeps may re-plan at a looser tolerance than the sign-off run.  Nothing already
 * computed changes. */
int pdn_set_solver_opts(pdn_ctx *ctx, double rtol, int32_t max_iter);

/* Same-side pairs (context created with PDN_TERMINAL_PAIRS).  side 0: bumps, side 1: loads.  out: DEVICE fp64,
 * nt*nt values (nt = n_bumps or n_loads), out[i*nt + j] = R_eff between terminals i and j of that side in the
 * whole 3D network (0 on the diagonal). */
int pdn_reff_same_side(pdn_ctx *ctx, int32_t side, double *out);

/* Eq. (4): bump `bump` (index into the create-time list) is held at v_bump, load k draws
 * i_load[k] (DEVICE, n_loads values, amperes); v_out[j] (DEVICE, n_loads values) receives the voltage of load j,
 *   v_j = v_bump - 1/2 sum_k i_load[k] (R_{b,j} + R_{b,k} - R_{j,k}).   Needs PDN_TERMINAL_PAIRS. */
int pdn_load_voltages(pdn_ctx *ctx, int32_t bump, const double *i_load, double v_bump, double *v_out);

/* The same Eq. (4), same arguments and result, for callers that must not allocate (code under CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc): pdn_load_voltages takes its scratch (R_b: n_loads values, R_LL:
 * n_loads^2 values, index lists) from the device pool, which may call cudaMalloc; this entry point keeps it in a
 * static __device__ array inside the library -- (PDN_STATIC_MAX_LOADS^2 + PDN_STATIC_MAX_LOADS) doubles = 2.0 MiB that
 * every GPU which loads libpdn.so holds until the process exits -- and calls no cudaMalloc, cudaFree or any
 * allocating routine (the first call on a device resolves the array's device address with cudaGetSymbolAddress).
 * n_loads > PDN_STATIC_MAX_LOADS: PDN_E_ARG, nothing launched (use pdn_load_voltages).  i_load, v_out: DEVICE, as above,
 * caller-owned.  The scratch is shared by ALL calls on a device and keeps the last call's contents; every word a call
 * reads it has written itself first, so nothing needs clearing -- but two calls whose kernels overlap on the GPU (two
 * contexts on different streams, two host threads) race: serialise them.  Work is ordered on the context's stream and
 * complete on return; if that stream is being captured the call records its three kernels and returns without
 * synchronising. */
#define PDN_STATIC_MAX_LOADS 512
int pdn_load_voltages_static(pdn_ctx *ctx, int32_t bump, const double *i_load, double v_bump, double *v_out);

/* Arbitrary-tier endpoints: R_eff in the whole 3D network between ANY nodes, on any
 * tier, of an existing context (any flags).  nodes: HOST array of n_nodes probes (duplicates allowed).  out:
 * DEVICE fp64, n_nodes*n_nodes values, out[a*n_nodes + b] = R_eff(node a, node b), 0 on the diagonal.
 * Cost: one port solve per probe on its own tier (full tolerance, gathered at the tier's TSV ends and at the
 * other probes of that tier), then one substitution with the factor of C kept since pdn_create / the last
 * pdn_update_tsvs (Eq. (18)-(22) PAPER.md:179-204 with the source / sink on arbitrary tiers; DESIGN.md
 * section 1).  The context is not changed.  On a sharded context (after pdn_finish) every rank that calls it
 * does all the probe solves itself. */
typedef struct pdn_node {
    int32_t tier, y, x;
} pdn_node;
int pdn_reff_nodes(pdn_ctx *ctx, int32_t n_nodes, const pdn_node *nodes, double *out);

/* One source against many nodes -- the R_eff map of Fig. 6(d).  src: HOST, one node; nodes: HOST
 * array of n_nodes probes on any tiers (duplicates and the source itself allowed); out: DEVICE fp64, n_nodes values,
 * out[a] = R_eff(src, nodes[a]) in the whole 3D network.  Same algebra as pdn_reff_nodes, but only one row and the
 * diagonal of its matrix are formed: on every tier that holds probes the TSV-port solves are repeated with the probes
 * in the gather list (by reciprocity they deliver Z_t[TSV port, probe]), every probe costs one DIAGONAL solve (loose
 * tolerance, second-order accurate like the bump / load solves of pdn_create), and the kept factor of C is applied
 * once to all n_nodes + 1 columns.  Memory is O((P + q_t) n_nodes) instead of pdn_reff_nodes' O(n_nodes^2), so a map
 * over every node of a tier is possible (it costs about one diagonal solve per node).  The context is not changed. */
int pdn_reff_from(pdn_ctx *ctx, const pdn_node *src, int32_t n_nodes, const pdn_node *nodes, double *out);

/* NEXT-4: one network sharded over several GPUs, one process per GPU.  The port solves of
 * a tier are independent, so with opts->shard_world = W > 1 pdn_create (same arguments on every
 * rank) imports all tiers but solves only slice opts->shard_rank of each tier's TSV sources and of its bump / load
 * sources -- contiguous, rank r owning [floor(r k / W), floor((r+1) k / W)) of k sources -- and returns an OPEN
 * context: pdn_reff & co. fail with PDN_E_ARG until pdn_finish.  The caller then makes every rank's rows present
 * on every rank (one broadcast per rank and tier over NCCL / NVLink: rows [tsv0, tsv0+ntsv) of the port matrix are
 * contiguous, ld doubles each; zdiag[term0 .. term0+nterm) likewise; with PDN_TERMINAL_PAIRS also rows
 * [ntsv_total+term0, ...)) and calls pdn_finish, which runs S2-S3 (replicated: milliseconds).
 * pdn_shard_slice: the slice of `rank` in `tier` (all zeros for a tier every rank reduced whole: uniform tiers,
 * meshes with n <= 4).  pdn_shard_buffers: DEVICE pointers of the tier's port matrix (ld = its leading dimension =
 * port count; ntsv_total = its number of TSV ports) and of zdiag. */
int pdn_shard_slice(const pdn_ctx *ctx, int32_t tier, int32_t rank, int32_t *tsv0, int32_t *ntsv, int32_t *term0,
                    int32_t *nterm);
int pdn_shard_buffers(pdn_ctx *ctx, int32_t tier, double **zt, int64_t *ld, int32_t *ntsv_total, double **zdiag);
int pdn_finish(pdn_ctx *ctx);

/* NULL-safe; frees all device and host memory of ctx. */
void pdn_destroy(pdn_ctx *ctx);

/* Device blocks released by pdn_destroy are kept in a process-wide cache and reused by the next
 * pdn_create (cudaMalloc / cudaFree of multi-GB workspaces cost tens of ms).  This returns them to
 * the driver.  Safe to call at any time from the thread that owns the contexts. */
void pdn_release_cache(void);

/* Helpers. */
const char *pdn_strerror(int status);
const char *pdn_last_error(void);                       /* last CUDA error string of this thread  */
int pdn_get_stats(const pdn_ctx *ctx, pdn_stats *out);

/* Port matrix of one tier (the intra-die array of PAPER.md:218): q = pdn_port_count(ctx, tier);
 * out (HOST, q*q doubles, row-major) receives Z_t = L_t^+ restricted to ports(t), where
 * ports(t) = [lower ends of interface t-1] ++ [upper ends of interface t] ++ [bumps if t = 0]
 * ++ [loads if t = d-1].  The intra-die effective resistance is R_jk = Z_jj + Z_kk - 2 Z_jk.
 * Entries between two bump/load ports other than the diagonal are not computed (NaN) unless the context was
 * created with PDN_TERMINAL_PAIRS: the bump x load method never needs them. */
int32_t pdn_port_count(const pdn_ctx *ctx, int32_t tier);
int pdn_get_port_matrix(const pdn_ctx *ctx, int32_t tier, double *out);

#ifdef __cplusplus
}
#endif
#endif /* PDN_H_ */
