// Microbenchmark behind DESIGN.md section 6: HBM read bandwidth of a pure bulk-async (TMA) stream, 148 CTAs, by tile size and
// ring depth (= bytes in flight per SM).  It is the ceiling for the way the contraction kernels read Phi.
// Build and run (one B200):  nvcc -std=c++17 -O3 -gencode arch=compute_100a,code=sm_100a -o tma_stream tma_stream.cu && ./tma_stream
// Output of round 1: profiles/r1_microbench.md.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#include "../csrc/tc_ptx.cuh"
// each CTA streams its contiguous share of a big buffer through an n-stage ring of `tile` bytes with 1-D bulk async copies
__global__ void __launch_bounds__(64, 1) stream(const uint8_t* src, size_t bytes_per_cta, int tile, int stages, int interleave, unsigned long long* sink) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint64_t full[16];
    if (threadIdx.x == 0) { for (int i = 0; i < stages; ++i) tc::mbar_init(&full[i], 1); tc::fence_barrier_init(); }
    __syncthreads();
    const size_t ntiles = bytes_per_cta / tile;
    // interleave = 0: CTA c reads [c*share, (c+1)*share); 1: tile t of CTA c is global tile t*grid + c
    auto addr = [&](size_t t) { return interleave ? src + (t * gridDim.x + blockIdx.x) * (size_t)tile : src + blockIdx.x * bytes_per_cta + t * (size_t)tile; };
    if (threadIdx.x == 0) {
        uint32_t ph = 0; int s = 0;
        for (size_t t = 0; t < (size_t)stages && t < ntiles; ++t) {
            tc::mbar_arrive_expect_tx(&full[t], tile);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(tc::smem_u32(smem + t * tile)), "l"(addr(t)), "r"(tile), "r"(tc::smem_u32(&full[t])) : "memory");
        }
        unsigned long long acc = 0;
        for (size_t t = 0; t < ntiles; ++t) {
            tc::mbar_wait(&full[s], ph);
            acc += *reinterpret_cast<volatile unsigned int*>(smem + s * tile);
            if (t + stages < ntiles) {
                tc::mbar_arrive_expect_tx(&full[s], tile);
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(tc::smem_u32(smem + s * tile)), "l"(addr(t + stages)), "r"(tile), "r"(tc::smem_u32(&full[s])) : "memory");
            }
            if (++s == stages) { s = 0; ph ^= 1; }
        }
        if (acc == 0x123456789ull) *sink = acc;
    }
}
int main() {
    const size_t total = 8ull << 30;
    uint8_t* d; cudaMalloc(&d, total); cudaMemset(d, 1, total);
    unsigned long long* sink; cudaMalloc(&sink, 8);
    cudaFuncSetAttribute(stream, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int inter : {0, 1}) for (int tile : {16384, 32768}) for (int stages : {2, 3, 4, 6, 8, 12}) {
        if ((size_t)tile * stages > 196608) continue;
        const int grid = 148;
        size_t per = (total / grid / tile) * tile;
        stream<<<grid, 64, tile * stages>>>(d, per, tile, stages, inter, sink);
        cudaEventRecord(e0);
        stream<<<grid, 64, tile * stages>>>(d, per, tile, stages, inter, sink);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        printf("%s tile %5d B stages %2d (%3d KB in flight/SM): %7.1f GB/s  %s\n", inter ? "interleaved" : "contiguous ", tile, stages, tile * stages / 1024, per * grid / (ms * 1e-3) / 1e9, cudaGetErrorString(cudaGetLastError()));
    }
    return 0;
}
