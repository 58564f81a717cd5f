// Microbenchmark behind DESIGN.md section 6: tensor-pipe cycles per tcgen05.mma.kind::tf32 instruction (M = 128) by operand
// form (A from tensor memory / shared memory), N, accumulator rotation and number of tcgen05.commit per 8 MMAs.
// Build and run (one B200):  nvcc -std=c++17 -O3 -gencode arch=compute_100a,code=sm_100a -o mma_cost mma_cost.cu && ./mma_cost
// Operands are arbitrary bits: only the timing is read.  Output of round 1: profiles/r1_microbench.md.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#include "../csrc/tc_ptx.cuh"
template <int variant>
__global__ void __launch_bounds__(128, 1) bench(int iters, long long* out) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint64_t bar; __shared__ uint64_t bars[4]; __shared__ uint32_t tbase;
    float* f = reinterpret_cast<float*>(smem);
    for (int i = threadIdx.x; i < 48 * 1024 / 4; i += 128) f[i] = 1.0f + (i % 7) * 0.125f;
    if (threadIdx.x == 0) { tc::mbar_init(&bar, 1); for (int i = 0; i < 4; ++i) tc::mbar_init(&bars[i], 1); tc::fence_barrier_init(); }
    if (threadIdx.x < 32) tc::tmem_alloc(&tbase, 512);
    tc::fence_proxy_async_smem();
    tc::tcgen05_fence_before(); __syncthreads(); tc::tcgen05_fence_after();
    const uint32_t tb = tbase;
    {   // init A region in TMEM cols 384..511 and D = 0
        uint32_t z[16]; for (int i = 0; i < 16; ++i) z[i] = __float_as_uint(1.0f);
        const uint32_t la = tb + ((uint32_t)((threadIdx.x >> 5) * 32) << 16);
        for (int c = 0; c < 512; c += 16) tc::tmem_st16(la + c, z);
        tc::tmem_st_wait();
    }
    tc::tcgen05_fence_before(); __syncthreads(); tc::tcgen05_fence_after();
    if (threadIdx.x < 32) {
        const uint64_t bdesc = tc::umma_desc_k_sw128(tc::smem_u32(smem));
        const uint64_t adesc = tc::umma_desc_k_sw128(tc::smem_u32(smem + 32 * 1024));
        const uint32_t id192 = tc::umma_idesc(2u, 128, 192), id96 = tc::umma_idesc(2u, 128, 96), id256 = tc::umma_idesc(2u, 128, 256);
        const uint32_t id48 = tc::umma_idesc(2u, 128, 48), id128 = tc::umma_idesc(2u, 128, 128);
        long long t0 = clock64();
        int n_instr = 0;
        for (int it = 0; it < iters; ++it) {
            if (tc::elect_one()) {
#pragma unroll
                for (int kk = 0; kk < 16; ++kk) {
                    const int k = kk & 3;
                    const uint32_t a = tb + 384 + k * 8;
                    const uint64_t b = bdesc + 2 * k;
                    switch (variant) {
                        case 0: tc::umma_tf32_ts(tb, a, b, id192, 1u); tc::umma_tf32_ts(tb + 96, a + 32, b, id96, 1u); break;
                        case 1: { uint32_t d = tb + ((it & 1) ? 192 : 0); tc::umma_tf32_ts(d, a, b, id192, 1u); tc::umma_tf32_ts(d + 96, a + 32, b, id96, 1u); } break;
                        case 2: tc::umma_tf32_ts(tb, a, b, id192, 1u); break;
                        case 3: tc::umma_tf32_ts(tb, a, b, id96, 1u); break;
                        case 4: tc::umma_tf32_ts(tb + (k & 3) * 96, a, b, id96, 1u); break;
                        case 5: tc::umma_tf32(tb, adesc + 2 * k, b, id96, 1u); break;
                        case 6: tc::umma_tf32(tb, adesc + 2 * k, b, id192, 1u); break;
                        case 7: tc::umma_tf32_ts(tb, a, b, id256, 1u); break;
                        case 8: tc::umma_tf32(tb, adesc + 2 * k, b, id256, 1u); break;
                        case 9: tc::umma_tf32_ts(tb, a, b, id192, 1u); tc::umma_tf32_ts(tb + 192, a + 32, b, id96, 1u); break;   // disjoint D columns
                        case 10: tc::umma_tf32_ts(tb, a, b, id48, 1u); break;
                        case 11: tc::umma_tf32_ts(tb, a, b, id128, 1u); break;
                        case 12: tc::umma_tf32(tb + (k & 3) * 96, adesc + 2 * k, b, id96, 1u); break;
                        case 13: case 14: case 15: case 16: tc::umma_tf32_ts(tb, a, b, id192, 1u); tc::umma_tf32_ts(tb + 96, a + 32, b, id96, 1u);
                            if (k == 3) { if (variant >= 14) tc::umma_commit(&bars[0]); if (variant >= 15) tc::umma_commit(&bars[1]); if (variant >= 16) tc::umma_commit(&bars[2]); } break;
                    }
                }
            }
            __syncwarp();
        }
        if (tc::elect_one()) tc::umma_commit(&bar);
        __syncwarp();
        tc::mbar_wait(&bar, 0);
        long long t1 = clock64();
        n_instr = iters * 16 * ((variant <= 1 || variant == 9 || variant >= 13) ? 2 : 1);
        if (threadIdx.x == 0 && blockIdx.x == 0) { out[0] = t1 - t0; out[1] = n_instr; }
    }
    __syncthreads();
    if (threadIdx.x < 32) { tc::tcgen05_fence_after(); tc::tmem_dealloc(tb, 512); }
}
int main() {
    long long* d; cudaMalloc(&d, 16);
    const char* names[] = {"TS wide192+one96 same D (current)", "TS wide+one alternating D regions", "TS N=192 same D", "TS N=96 same D", "TS N=96 rotating 4 D", "SS N=96 same D", "SS N=192 same D", "TS N=256 same D", "SS N=256 same D", "TS wide192 + one96 disjoint D", "TS N=48", "TS N=128", "SS N=96 rotating 4 D", "cur pattern, no commit", "cur + 1 commit / 8 MMAs", "cur + 2 commits / 8 MMAs", "cur + 3 commits / 8 MMAs"};
    auto run = [&](auto kern, int v) {
        long long h[2];
        kern<<<148, 128, 64 * 1024>>>(500, d); cudaDeviceSynchronize();
        kern<<<148, 128, 64 * 1024>>>(500, d);
        cudaError_t e = cudaDeviceSynchronize();
        cudaMemcpy(h, d, 16, cudaMemcpyDeviceToHost);
        printf("%-40s %s  cycles/instr %.1f\n", names[v], cudaGetErrorString(e), (double)h[0] / h[1]);
    };
#define RUN(V) cudaFuncSetAttribute(bench<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024); run(bench<V>, V);
    RUN(0) RUN(1) RUN(2) RUN(3) RUN(4) RUN(5) RUN(6) RUN(7) RUN(8) RUN(9) RUN(10) RUN(11) RUN(12) RUN(13) RUN(14) RUN(15) RUN(16)
    return 0;
}
