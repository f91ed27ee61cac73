// Host-side runtime of libpdn: error plumbing, the device-memory pool and RAII buffers, the context, launch
// bookkeeping (counts, per-class CUDA-event timers) and TMA descriptor encoding.  Included by pdn_api.cu only.
#pragma once

using namespace pdn;

namespace {

thread_local std::string g_last_error;

struct CudaFail {
    cudaError_t e;
    const char* what;
};

#define CK(call)                                                    \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) throw CudaFail{e__, #call};         \
    } while (0)

struct StatusFail {
    int status;
    std::string msg;
};

// kernel classes for the per-class timers / byte model
enum { KC_PQ = 0, KC_DOWN0, KC_UP0, KC_DOWNC, KC_UPC, KC_SMALL, KC_DENSE, KC_PAIR, KC_COUNT };

// ------------------------------------------------------------------------------------------------
// Device memory: a process-wide cache of freed blocks.  pdn_create needs tens of GB of workspace;
// cudaMalloc / cudaFree of blocks that size cost tens of milliseconds each, so released blocks are
// kept and handed out again (best fit within 25 %).  pdn_release_cache() returns them to the driver;
// an allocation failure does so automatically before giving up.
struct DevPool {
    static constexpr int MAX_DEV = 64;
    std::mutex mu;
    std::multimap<size_t, void*> free_blocks[MAX_DEV];  // per device: a block only ever goes back to its own device
    size_t cached[MAX_DEV] = {};

    static int current_device() {
        int dev = 0;
        cudaGetDevice(&dev);
        return dev & (MAX_DEV - 1);
    }
    void* get(size_t n, int dev) {
        {
            std::lock_guard<std::mutex> g(mu);
            auto& fb = free_blocks[dev];
            auto it = fb.lower_bound(n);
            if (it != fb.end() && it->first <= n + n / 4 + 4096) {
                void* p = it->second;
                cached[dev] -= it->first;
                fb.erase(it);
                return p;
            }
        }
        void* p = nullptr;
        cudaError_t e = cudaMalloc(&p, n);
        if (e != cudaSuccess) {
            cudaGetLastError();
            trim();
            e = cudaMalloc(&p, n);
            if (e != cudaSuccess) { cudaGetLastError(); return nullptr; }
        }
        return p;
    }
    void put(void* p, size_t n, int dev) {
        std::lock_guard<std::mutex> g(mu);
        free_blocks[dev].emplace(n, p);
        cached[dev] += n;
    }
    void trim() {
        std::lock_guard<std::mutex> g(mu);
        for (int d = 0; d < MAX_DEV; ++d) {
            for (auto& kv : free_blocks[d]) cudaFree(kv.second);
            free_blocks[d].clear();
            cached[d] = 0;
        }
    }
    size_t cached_bytes(int dev) {
        std::lock_guard<std::mutex> g(mu);
        return cached[dev];
    }
};
DevPool g_pool;

// Pinned host scratch for the per-iteration read-backs: blocks are kept for the life of the process and handed
// from one workspace to the next (cudaMallocHost / cudaFreeHost stall for hundreds of ms now and then); a
// workspace owns its block while it lives, so host threads solving tiers concurrently never share one.
struct PinnedPool {
    std::mutex mu;
    std::vector<std::pair<size_t, void*>> free_blocks;
    void* get(size_t n, size_t* got) {
        {
            std::lock_guard<std::mutex> g(mu);
            for (size_t i = 0; i < free_blocks.size(); ++i)
                if (free_blocks[i].first >= n) {
                    void* p = free_blocks[i].second;
                    *got = free_blocks[i].first;
                    free_blocks.erase(free_blocks.begin() + i);
                    return p;
                }
        }
        void* p = nullptr;
        n = std::max<size_t>(n, 16384);
        if (cudaMallocHost(&p, n) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        *got = n;
        return p;
    }
    void put(void* p, size_t n) {
        std::lock_guard<std::mutex> g(mu);
        free_blocks.emplace_back(n, p);
    }
};
PinnedPool g_pinned;

// PDN_POISON=1 in the environment (read once): every device block handed out is first filled with 0xFF bytes --
// NaN as a double or float, -1 as an int -- so that any read of memory the library did not write itself turns
// up as a NaN in the results (PDN_E_NUMERIC / a failed parity test) instead of depending on what the block held
// before.  A debugging aid (the pool recycles blocks, which hides such reads); compute-sanitizer's initcheck is
// not available on every box.
inline bool poison_enabled() {
    static const bool on = [] { const char* e = getenv("PDN_POISON"); return e && e[0] && e[0] != '0'; }();
    return on;
}

struct DevBuf {  // RAII device allocation on the device that is current at alloc()
    void* p = nullptr;
    size_t bytes = 0;
    int dev = 0;
    DevBuf() = default;
    DevBuf(const DevBuf&) = delete;
    DevBuf& operator=(const DevBuf&) = delete;
    DevBuf(DevBuf&& o) noexcept : p(o.p), bytes(o.bytes), dev(o.dev) { o.p = nullptr; o.bytes = 0; }
    DevBuf& operator=(DevBuf&& o) noexcept {
        if (this != &o) { release(); p = o.p; bytes = o.bytes; dev = o.dev; o.p = nullptr; o.bytes = 0; }
        return *this;
    }
    ~DevBuf() { release(); }
    void release() { if (p) g_pool.put(p, bytes, dev); p = nullptr; bytes = 0; }
    void alloc(size_t n) {
        release();
        n = n < 256 ? 256 : (n + 255) & ~size_t(255);
        dev = DevPool::current_device();
        p = g_pool.get(n, dev);
        if (!p) throw StatusFail{PDN_E_NOMEM, "cudaMalloc of " + std::to_string(n) + " bytes failed"};
        bytes = n;
        if (poison_enabled()) { CK(cudaMemset(p, 0xFF, n)); CK(cudaDeviceSynchronize()); }
    }
    template <class T> T* as() const { return static_cast<T*>(p); }
};

struct TierPorts {
    int ntsv = 0, nterm = 0, q = 0;   // TSV ports, terminal ports, total
    int nrows = 0;                    // rows of ZT: ntsv, or q when the terminal rows are kept (PDN_TERMINAL_PAIRS)
    std::vector<int> node;            // pitched offset y*pitch + x of every port, port order of port.cuh
    DevBuf d_node;                    // device copy
    DevBuf ZT;                        // nrows x q
    DevBuf zdiag;                     // nterm
    DevBuf gx0, gy0;                  // sanitised pitched level-0 planes, kept for pdn_update_tsvs
    bool whole = false;               // reduced whole on this rank (uniform tier, n <= 4): nothing to exchange
};

}  // namespace

struct pdn_ctx {
    int d = 0, n = 0, m = 0, nl = 0, p0 = 0;
    int device = 0;                   // the CUDA device the context lives on (current at pdn_create)
    std::vector<int> p;               // TSVs per interface
    std::vector<std::vector<double>> rt;
    std::vector<std::vector<int>> site;   // per interface: pitched offsets of the TSV sites, in list order
    std::vector<int> bump_id, load_id;    // pitched offsets of the terminals
    cudaStream_t stream = nullptr;
    pdn_opts opts{};
    std::vector<TierPorts> tiers;
    DevBuf A1, X0, u, w;              // operands of the pair kernel
    struct Side { DevBuf A, X, ys, t; int p = 0; } side[2];  // same-side pairs: [0] bumps, [1] loads (PDN_TERMINAL_PAIRS)
    std::vector<DevBuf> Li, Vf, KB;   // factor of C kept for pdn_reff_nodes: L_i^-1, L_{i-1}^-1 K_{i-1,i}, (K^-1 B)_i
    DevBuf Sinv;                      // inverse of the Schur complement B^T K^-1 B ((d-1)^2)
    bool terminal_pairs = false;
    bool nu_auto = true;                  // opts.nu was left at its default: strongly anisotropic tiers may deepen it
    int shard_rank = 0, shard_world = 1;  // NEXT-4
    bool open = false;                    // sharded context whose rows have not been completed / S2-S3 not run
    bool poisoned = false;                // pdn_update_tsvs failed after its commit point: only pdn_destroy is left
    pdn_stats stats{};
    double class_ms[KC_COUNT] = {};
    double class_bytes[KC_COUNT] = {};
    int64_t class_launches[KC_COUNT] = {};
    std::mutex mu;                        // guards the counters below when tiers are solved by several host threads
    bool time_kernels = false;
    bool debug = false;                   // PDN_DEBUG was set in the environment at pdn_create: iteration history on stderr
    std::vector<std::pair<int, std::pair<cudaEvent_t, cudaEvent_t>>> pending_events;
    std::vector<cudaEvent_t> event_pool;
};

namespace {

// ------------------------------------------------------------------------------------------------
// launch bookkeeping: every kernel goes through Launcher::run so that launches are counted and,
// with PDN_TIME_KERNELS, bracketed by CUDA events on the launching stream.
struct Launcher {
    pdn_ctx* c;
    cudaStream_t s;
    cudaEvent_t get_event() {
        if (!c->event_pool.empty()) { cudaEvent_t e = c->event_pool.back(); c->event_pool.pop_back(); return e; }
        cudaEvent_t e;
        CK(cudaEventCreate(&e));
        return e;
    }
    template <class F>
    void run(int cls, double bytes, F&& f) {
        cudaEvent_t a = nullptr, b = nullptr;
        if (c->time_kernels) {
            { std::lock_guard<std::mutex> g(c->mu); a = get_event(); b = get_event(); }
            CK(cudaEventRecord(a, s));
        }
        f();
        CK(cudaGetLastError());
        if (c->time_kernels) CK(cudaEventRecord(b, s));
        std::lock_guard<std::mutex> g(c->mu);
        if (c->time_kernels) c->pending_events.push_back({cls, {a, b}});
        c->class_launches[cls]++;
        c->class_bytes[cls] += bytes;
        c->stats.kernel_launches++;
        if (cls <= KC_SMALL) c->stats.stencil_launches++;
    }
    void resolve() {  // call after a stream synchronise
        for (auto& pe : c->pending_events) {
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, pe.second.first, pe.second.second));
            c->class_ms[pe.first] += ms;
            c->event_pool.push_back(pe.second.first);
            c->event_pool.push_back(pe.second.second);
        }
        c->pending_events.clear();
    }
};

// Runs `set` once per device (kernel attributes are per device); the bit is published after the attributes are
// in place, so a second host thread either sees it set or sets the same attributes again (harmless).
template <class F>
inline void once_per_device(std::atomic<uint64_t>& mask, F&& set) {
    const uint64_t bit = 1ull << DevPool::current_device();
    if (mask.load(std::memory_order_acquire) & bit) return;
    set();
    mask.fetch_or(bit, std::memory_order_release);
}

inline unsigned cdiv(size_t a, size_t b) { return (unsigned)((a + b - 1) / b); }
// gridDim.y of the kernels that walk a problem dimension with `for (row = blockIdx.y; row < rows; row += gridDim.y)`
inline unsigned grid_rows(size_t rows) { return (unsigned)std::min<size_t>(std::max<size_t>(rows, 1), 65535); }

// ------------------------------------------------------------------------------------------------
// TMA descriptors: a batched pitched vector v[B][ny][pitch] as a 3D tensor (x, y, b) of doubles whose
// x extent is the true nx (so pad columns read as zeros) and a box of bx x by x 1.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres));
        if (!p || qres != cudaDriverEntryPointSuccess) throw StatusFail{PDN_E_CUDA, "cuTensorMapEncodeTiled is not available"};
        fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

CUtensorMap make_map(const void* base, int nx, int ny, int pitch, int B, int box_x, int box_y) {
    CUtensorMap m;
    const cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)B};
    const cuuint64_t strides[2] = {(cuuint64_t)pitch * 8, (cuuint64_t)pitch * ny * 8};
    const cuuint32_t box[3] = {(cuuint32_t)box_x, (cuuint32_t)box_y, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = encode_tiled_fn()(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), dims, strides,
                                         box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) throw StatusFail{PDN_E_CUDA, "cuTensorMapEncodeTiled failed with code " + std::to_string((int)r)};
    return m;
}

// A pitched FP32 matrix (rows x cols, row pitch `pitch` floats) as a 2D tensor with a box of box_x x box_y.
CUtensorMap make_map_2d_f32(const void* base, int cols, int rows, int pitch, int box_x, int box_y) {
    CUtensorMap m;
    const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)pitch * 4};
    const cuuint32_t box[2] = {(cuuint32_t)box_x, (cuuint32_t)box_y};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode_tiled_fn()(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), dims, strides,
                                         box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) throw StatusFail{PDN_E_CUDA, "cuTensorMapEncodeTiled (2D) failed with code " + std::to_string((int)r)};
    return m;
}
}  // namespace
