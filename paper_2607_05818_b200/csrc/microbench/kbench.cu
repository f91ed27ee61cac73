// Developer microbenchmark (not part of libpdn.so): times the level-0 stencil kernels of stencil3.cuh -- k_down3
// (fused and plain), k_up3, k_pq3 -- on dummy data, without the PCG around them, so that a kernel change can be
// judged in seconds.  The data are not a valid multigrid problem: nothing is checked here, parity is the job of
// tests/test_gpu_parity.py through the library.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -std=c++17 -diag-suppress 177 kbench.cu -o kbench -lcuda
//   ./kbench [n=1024] [rhs=512] [reps=5] [all|down|downc|up|pq]
//
// reps = 5 times cold, unthrottled launches; reps = 300-400 keeps the part busy for seconds, the 1000 W power cap
// pulls the SM clock to ~1.7 GHz and the averages land on what bench.py reports per kernel class (profiles/r2_microbench.md).
// -DKB_R / -DKB_W / -DKB_NU select patch rows, warps per block and smoothing steps of the V-cycle kernels.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>
#include "../common.cuh"
#include "../stencil3.cuh"

using namespace pdn;
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at %s:%d\n", cudaGetErrorString(e_), __FILE__, __LINE__); exit(1); } } while (0)

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn enc() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) { void* p = nullptr; cudaDriverEntryPointQueryResult q; CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q)); fn = (EncodeTiledFn)p; }
    return fn;
}
static CUtensorMap make_map(const void* base, int nx, int ny, int pitch, int B, int bx, int by) {
    CUtensorMap m;
    const cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)B};
    const cuuint64_t strides[2] = {(cuuint64_t)pitch * 8, (cuuint64_t)pitch * ny * 8};
    const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1};
    const cuuint32_t es[3] = {1, 1, 1};
    CUresult r = enc()(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { printf("encode failed %d\n", (int)r); exit(1); }
    return m;
}
static int rhs_per_block(int tiles, int B, int G, int cap) {
    const int sms = 148; const double setup = 2.0;
    int best = 1; double bc = 1e300;
    for (int g = 1; g <= std::min(G, cap); ++g) {
        long blocks = (long)tiles * ((B + g - 1) / g);
        double c = (double)((blocks + sms - 1) / sms) * (g + setup);
        if (c < bc) { bc = c; best = g; }
    }
    return best;
}
__global__ void k_fill(double* p, size_t n, double a, double b) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        p[i] = a + b * (double)((i * 2654435761u) & 1023) / 1024.0;
}
__global__ void k_fill_sc(float2* p, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        p[i] = make_float2(0.5f, 2.0f);
}

#ifndef KB_R
#define KB_R 6
#endif
#ifndef KB_W
#define KB_W 12
#endif
#ifndef KB_NU
#define KB_NU 4
#endif

int main(int argc, char** argv) {
    const int n = argc > 1 ? atoi(argv[1]) : 1024, B = argc > 2 ? atoi(argv[2]) : 512, reps = argc > 3 ? atoi(argv[3]) : 5;
    const int pitch = (n + 1) & ~1;
    const size_t plane = (size_t)n * pitch, vec = plane * B;
    const int nc = (n + 1) / 2, cpitch = (nc + 1) & ~1;
    const size_t cplane = (size_t)nc * cpitch;
    double *r0, *r1, *q, *y, *z, *p0, *p1, *rc, *e, *gx, *gy, *hE, *hS, *alpha, *acc;
    float2* sc;
    CK(cudaMalloc(&r0, vec * 8)); CK(cudaMalloc(&r1, vec * 8)); CK(cudaMalloc(&q, vec * 8)); CK(cudaMalloc(&y, vec * 8));
    CK(cudaMalloc(&z, vec * 8)); CK(cudaMalloc(&p0, vec * 8)); CK(cudaMalloc(&p1, vec * 8));
    CK(cudaMalloc(&rc, cplane * B * 8)); CK(cudaMalloc(&e, cplane * B * 8));
    CK(cudaMalloc(&gx, plane * 8)); CK(cudaMalloc(&gy, plane * 8)); CK(cudaMalloc(&hE, plane * 8)); CK(cudaMalloc(&hS, plane * 8));
    CK(cudaMalloc(&sc, plane * 8)); CK(cudaMalloc(&alpha, B * 8)); CK(cudaMalloc(&acc, 4 * B * 8));
    for (double* v : {r0, r1, q, y, z, p0, p1}) k_fill<<<2048, 256>>>(v, vec, -0.5, 1.0);
    k_fill<<<2048, 256>>>(rc, cplane * B, -0.5, 1.0); k_fill<<<2048, 256>>>(e, cplane * B, -0.5, 1.0);
    k_fill<<<512, 256>>>(gx, plane, 0.9, 0.2); k_fill<<<512, 256>>>(gy, plane, 0.9, 0.2);
    k_fill<<<512, 256>>>(hE, plane, 0.22, 0.05); k_fill<<<512, 256>>>(hS, plane, 0.22, 0.05);
    k_fill_sc<<<512, 256>>>(sc, plane);
    k_fill<<<4, 256>>>(alpha, B, 0.3, 0.1);
    CK(cudaMemset(acc, 0, 4 * B * 8));
    CK(cudaDeviceSynchronize());
    Level L{n, n, pitch, gx, gy, hE, hS, sc};
    ChebR ch{}; ch.nu = KB_NU;
    for (int k = 0; k < MAX_NU; ++k) ch.w[k] = 0.6 + 0.05 * k;
    constexpr int R = KB_R, W = KB_W, EH = R * W, NU = KB_NU, H = halo_of(NU);
    CUtensorMap m_r0 = make_map(r0, n, n, pitch, B, T3_EW, EH), m_q = make_map(q, n, n, pitch, B, T3_EW, EH), m_y = make_map(y, n, n, pitch, B, T3_EW, EH);
    CUtensorMap m_r1 = make_map(r1, n, n, pitch, B, T3_EW, EH), m_z = make_map(z, n, n, pitch, B, T3_EW, EH), m_p = make_map(p0, n, n, pitch, B, T3_EW, EH);
    CUtensorMap m_e = make_map(e, nc, nc, cpitch, B, T3_ECW, EH / 2);
    const size_t TILE = (size_t)EH * T3_EW * 8, SC = (size_t)EH * 32 * 16;
    cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    const double V = (double)B * n * n * 8.0;
    auto time_it = [&](const char* name, double bytes, auto&& launch) {
        for (int i = 0; i < 2; ++i) launch();
        CK(cudaDeviceSynchronize());
        float best = 1e30f, sum = 0.f;
        for (int i = 0; i < reps; ++i) {
            CK(cudaEventRecord(e0)); launch(); CK(cudaEventRecord(e1)); CK(cudaEventSynchronize(e1));
            float ms; CK(cudaEventElapsedTime(&ms, e0, e1)); best = std::min(best, ms); sum += ms;
        }
        CK(cudaGetLastError());
        printf("%-10s  avg %.3f ms  best %.3f ms   %.0f GB/s avg  %.0f GB/s best   (frac of 6552: %.3f)\n", name, sum / reps, best, bytes / (sum / reps) * 1e-6, bytes / best * 1e-6, bytes / (sum / reps) * 1e-6 / 6552.3);
    };
    const std::string which = argc > 4 ? argv[4] : "all";
    {   // down0 (fused)
        constexpr int IW = T3_EW - 2 * H, IH = EH - 2 * H;
        const int tx = (n + IW - 1) / IW, ty = (n + IH - 1) / IH, G = rhs_per_block(tx * ty, B, 64, T3_MAX_G);
        dim3 grid(tx, ty, (B + G - 1) / G);
        const size_t smem = 4 * TILE + SC + sizeof(Exch<W, double>);
        CK(cudaFuncSetAttribute(k_down3<R, W, NU, true, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (which == "all" || which == "down")
            time_it("down0", 4.25 * V, [&] { k_down3<R, W, NU, true, double><<<grid, 32 * W, smem>>>(m_r0, m_q, L, ch, alpha, r1, y, rc, nc, nc, cpitch, acc, B, G, nullptr); });
        const size_t smem2 = 2 * TILE + SC + sizeof(Exch<W, double>);
        CK(cudaFuncSetAttribute(k_down3<R, W, NU, false, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
        if (which == "all" || which == "downc")
            time_it("down_plain", 2.25 * V, [&] { k_down3<R, W, NU, false, double><<<grid, 32 * W, smem2>>>(m_r0, m_r0, L, ch, alpha, nullptr, y, rc, nc, nc, cpitch, acc, B, G, nullptr); });
        printf("   grid %d x %d x %d, G = %d, smem %zu\n", tx, ty, (B + G - 1) / G, G, smem);
    }
    {   // up0 (with dot)
        constexpr int IW = T3_EW - 2 * H, IH = EH - 2 * H;
        const int tx = (n + IW - 1) / IW, ty = (n + IH - 1) / IH, G = rhs_per_block(tx * ty, B, 64, T3_MAX_G);
        dim3 grid(tx, ty, (B + G - 1) / G);
        const size_t smem = 4 * TILE + 2 * Geom<R, W, 2>::ETILE_BYTES + SC + sizeof(Exch<W, double>);
        CK(cudaFuncSetAttribute(k_up3<R, W, NU, true, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (which == "all" || which == "up")
            time_it("up0", 3.25 * V, [&] { k_up3<R, W, NU, true, double><<<grid, 32 * W, smem>>>(m_r1, m_y, m_e, L, ch, z, acc + B, B, G, nullptr); });
        printf("   grid %d x %d x %d, G = %d, smem %zu\n", tx, ty, (B + G - 1) / G, G, smem);
    }
    {   // pq: w = L z, q = w + beta q (in place), z.w, sum(z)
        constexpr int PR = 12, PW = 6, IW = T3_EW - 4, IH = PR * PW - 4;
        const int tx = (n + IW - 1) / IW, ty = (n + IH - 1) / IH, G = rhs_per_block(tx * ty, B, 64, T3_MAX_G_PQ);
        dim3 grid(tx, ty, (B + G - 1) / G);
        const size_t smem = 5 * (size_t)PR * PW * T3_EW * 8 + sizeof(Exch<PW>);
        CUtensorMap mz = make_map(z, n, n, pitch, B, T3_EW, PR * PW), mq = make_map(q, n, n, pitch, B, T3_EW, PR * PW);
        CK(cudaFuncSetAttribute(k_pq3<PR, PW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (which == "all" || which == "pq")
            time_it("pq", 3.0 * V, [&] { k_pq3<PR, PW><<<grid, 32 * PW, smem>>>(mz, mq, L, alpha, q, acc + 2 * B, acc + 3 * B, B, G, nullptr, 0); });
    }
    return 0;
}
