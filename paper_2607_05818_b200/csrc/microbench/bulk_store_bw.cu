// Developer microbenchmark (not part of libpdn.so): per-SM throughput of asynchronous bulk stores shared -> global
// (cp.async.bulk.global.shared::cta, the copy-engine path).  Result on B200 (profiles/r2_microbench.md): 32 B/clk per
// SM as well (23 B/clk with 448-byte chunks): the copy engine does not widen the SM's store path, it only takes the
// stores off the LSU.    nvcc -gencode arch=compute_100a,code=sm_100a -O3 bulk_store_bw.cu -o bulk_store_bw && ./bulk_store_bw
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
// per-SM throughput of bulk async stores smem -> global (cp.async.bulk.global.shared::cta)
__global__ void __launch_bounds__(128, 1) k_bulk(double* out, size_t per_block_bytes, int chunk, int iters, long long* clk) {
    extern __shared__ __align__(128) unsigned char sm[];
    for (int i = threadIdx.x; i < chunk / 8; i += blockDim.x) reinterpret_cast<double*>(sm)[i] = (double)i;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    long long t0 = clock64();
    if (threadIdx.x == 0) {
        unsigned char* dst = reinterpret_cast<unsigned char*>(out) + (size_t)blockIdx.x * per_block_bytes;
        const uint32_t src = (uint32_t)__cvta_generic_to_shared(sm);
        for (int i = 0; i < iters; ++i) {
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst + (size_t)i * chunk), "r"(src), "r"(chunk) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 4;" ::: "memory");
        }
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
    __syncthreads();
    long long t1 = clock64();
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}
int main() {
    const int nb = 148;
    long long* c; cudaMalloc(&c, nb * 8);
    long long h[148];
    for (int chunk : {448, 4096, 28672}) {
        const int iters = (32 << 20) / chunk;
        const size_t per_block = (size_t)iters * chunk;
        double* d; cudaMalloc(&d, nb * per_block);
        cudaFuncSetAttribute(k_bulk, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
        for (int blocks : {1, 148}) {
            k_bulk<<<blocks, 128, 32768>>>(d, per_block, chunk, iters, c); cudaDeviceSynchronize();
            cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
            cudaEventRecord(e0); k_bulk<<<blocks, 128, 32768>>>(d, per_block, chunk, iters, c); cudaEventRecord(e1); cudaEventSynchronize(e1);
            float ms; cudaEventElapsedTime(&ms, e0, e1);
            cudaMemcpy(h, c, blocks * 8, cudaMemcpyDeviceToHost);
            printf("bulk store chunk %5d B, blocks %3d: %.1f B/clk/SM (block 0), total %.0f GB/s  (%s)\n", chunk, blocks, (double)per_block / h[0], blocks * per_block / ms * 1e-6, cudaGetErrorString(cudaGetLastError()));
        }
        cudaFree(d);
    }
    return 0;
}
