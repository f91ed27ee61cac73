// Developer microbenchmark (not part of libpdn.so): how fast ONE SM can store to / load from global memory with
// 16-byte accesses, alone and with all 148 SMs busy.  Result on B200 (profiles/r2_microbench.md): STG.128 drains at
// 32.0 B/clk per SM whatever the cache hint, LDG.128 at ~108 B/clk -- the store side is what the output phases of the
// V-cycle kernels wait for.    nvcc -gencode arch=compute_100a,code=sm_100a -O3 store_bw.cu -o store_bw && ./store_bw
#include <cstdio>
#include <cuda_runtime.h>
__global__ void __launch_bounds__(384, 1) k_st(double* out, size_t per_block, int iters, long long* clk) {
    double2* p = reinterpret_cast<double2*>(out + (size_t)blockIdx.x * per_block) + threadIdx.x;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) { *p = make_double2((double)i, 1.0); p += 384; }
    long long t1 = clock64();
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}
__global__ void __launch_bounds__(384, 1) k_ld(const double* in, size_t per_block, int iters, long long* clk, double* sink) {
    const double2* p = reinterpret_cast<const double2*>(in + (size_t)blockIdx.x * per_block) + threadIdx.x;
    long long t0 = clock64();
    double a = 0;
    for (int i = 0; i < iters; i += 4) { double2 v0 = p[0], v1 = p[384], v2 = p[768], v3 = p[1152]; a += v0.x + v1.y + v2.x + v3.y; p += 4 * 384; }
    long long t1 = clock64();
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
    if (a == 1.2345) *sink = a;
}
int main() {
    const int nb = 148, iters = 4096; const size_t per_block = (size_t)iters * 384 * 2;
    double* d; long long* c; cudaMalloc(&d, nb * per_block * 8); cudaMalloc(&c, nb * 8); cudaMemset(d, 0, nb * per_block * 8);
    long long h[148];
    for (int blocks : {1, 16, 74, 148}) {
        k_st<<<blocks, 384>>>(d, per_block, iters, c); cudaDeviceSynchronize();
        cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
        cudaEventRecord(e0); k_st<<<blocks, 384>>>(d, per_block, iters, c); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        cudaMemcpy(h, c, blocks * 8, cudaMemcpyDeviceToHost);
        printf("STG.128 blocks %3d: %.1f B/clk/SM (block 0), total %.0f GB/s\n", blocks, (double)per_block * 8 / h[0], blocks * per_block * 8 / ms * 1e-6);
        cudaEventRecord(e0); k_ld<<<blocks, 384>>>(d, per_block, iters, c, d); cudaEventRecord(e1); cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        cudaMemcpy(h, c, blocks * 8, cudaMemcpyDeviceToHost);
        printf("LDG.128 blocks %3d: %.1f B/clk/SM (block 0), total %.0f GB/s\n", blocks, (double)per_block * 8 / h[0], blocks * per_block * 8 / ms * 1e-6);
    }
    return 0;
}
