// admm_phit_apply_static: the dose-rate contraction of Eq. (6) (W = G . Phi) for callers that may not allocate
// (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  It is a variant of the split-K cross-check kernel
// (simt_contract_kernel<EPI_K1_PARTIAL> in kernels.cu, whose partial sums live in the handle's cudaMalloc'ed d_partial): here the
// partial sums and the arrival tickets live in ONE file-scope __device__ array of ADMM_STATIC_SCRATCH_BYTES, and the block that
// arrives last at an output tile adds the partials in split order (fp64) -- one launch, no handle, no allocation.
//
// This file is self-contained on purpose: it shares no state with the handle-based path and changes none of it.
#include "../../include/admm_b200.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <mutex>

namespace {

constexpr int kTile = 64;                       // output tile: 64 time variables x 64 plans, 256 threads, 4 x 4 outputs each
constexpr int kKStep = 16;                      // k-slice staged in shared memory
constexpr int kMaxSplits = 64;
constexpr int64_t kTicketWords = 4096;          // one arrival counter per output tile, at the head of the scratch array
constexpr int64_t kPartialFloats = ((int64_t)ADMM_STATIC_SCRATCH_BYTES - kTicketWords * 4) / 4;
constexpr int kMaxDevices = 64;

// The scratch.  In HOST code this name is a stand-in, not a device address: the address comes from cudaGetSymbolAddress below.
static __device__ __align__(256) unsigned char g_static_scratch[ADMM_STATIC_SCRATCH_BYTES];

// W[q][m] = sum_i G[q][i] Phi[i][m];  Phi [N][ld] row-major, G [B][ld_g], W [B][n] fp64.
// grid (ceil(n/64), ceil(B/64), splits); split z covers points [z k_per_split, (z+1) k_per_split).
__global__ void __launch_bounds__(256) phit_apply_static_kernel(const float* __restrict__ phi, int64_t N, int64_t n, int64_t ld,
                                                                const float* __restrict__ g, int B, int64_t ld_g,
                                                                int64_t k_per_split, unsigned char* scratch,
                                                                double* __restrict__ w_out) {
    __shared__ float sX[kKStep][kTile + 1];
    __shared__ float sY[kKStep][kTile + 1];
    __shared__ int s_last;
    unsigned int* tickets = reinterpret_cast<unsigned int*>(scratch);
    float* partial = reinterpret_cast<float*>(scratch) + kTicketWords;
    const int splits = (int)gridDim.z, split = (int)blockIdx.z;
    const int64_t m0 = (int64_t)blockIdx.x * kTile;
    const int q0 = (int)blockIdx.y * kTile;
    const int64_t kbeg = (int64_t)split * k_per_split;
    const int64_t kend = (kbeg + k_per_split < N) ? kbeg + k_per_split : N;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float c[4][4] = {};
    for (int64_t k0 = kbeg; k0 < kend; k0 += kKStep) {
        for (int i = threadIdx.x; i < kKStep * kTile; i += 256) {
            {   // Phi: consecutive threads read consecutive time variables of one point (coalesced)
                const int r = i & (kTile - 1), kk = i >> 6;
                const int64_t k = k0 + kk, m = m0 + r;
                sX[kk][r] = (k < kend && m < n) ? phi[k * ld + m] : 0.f;
            }
            {   // G: consecutive threads read consecutive points of one plan
                const int kk = i & (kKStep - 1), r = i >> 4;
                const int64_t k = k0 + kk; const int q = q0 + r;
                sY[kk][r] = (k < kend && q < B) ? g[(int64_t)q * ld_g + k] : 0.f;
            }
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < kKStep; ++kk) {
            float xv[4], yv[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) { xv[a] = sX[kk][ty * 4 + a]; yv[a] = sY[kk][tx * 4 + a]; }
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) c[a][b] += xv[a] * yv[b];
        }
        __syncthreads();
    }
    // partial[split][q][m]
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int64_t m = m0 + ty * 4 + a; const int q = q0 + tx * 4 + b;
            if (m < n && q < B) __stcg(partial + ((int64_t)split * B + q) * n + m, c[a][b]);
        }
    __threadfence();
    __syncthreads();
    const unsigned int tile = blockIdx.y * gridDim.x + blockIdx.x;
    if (threadIdx.x == 0) s_last = (atomicAdd(tickets + tile, 1u) == (unsigned int)(splits - 1));
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // the last block to arrive adds the tile's partial sums, always in split order: the result does not depend on which block that is
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int64_t m = m0 + ty * 4 + a; const int q = q0 + tx * 4 + b;
            if (m >= n || q >= B) continue;
            double w = 0.0;
            for (int s = 0; s < splits; ++s) w += (double)__ldcg(partial + ((int64_t)s * B + q) * n + m);
            w_out[(int64_t)q * n + m] = w;
        }
    if (threadIdx.x == 0) tickets[tile] = 0u;         // leave the counter as the next call needs it
}

struct DeviceSlot {
    bool ready = false;
    unsigned char* scratch = nullptr;      // device address of g_static_scratch on this device
    int sm_count = 0;
};
std::mutex g_mu;
DeviceSlot g_slot[kMaxDevices];

void say(char* errbuf, int32_t len, const char* msg) {
    if (errbuf && len > 0) std::snprintf(errbuf, (size_t)len, "%s", msg);
}

bool on_device(const void* p, int device) {
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return (a.type == cudaMemoryTypeDevice && a.device == device) || a.type == cudaMemoryTypeManaged;
}

struct DeviceGuard {
    int prev = -1; bool switched = false;
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

}  // namespace

extern "C" admm_status admm_phit_apply_static(const float* phi, int64_t N, int64_t n, int64_t ld, const float* g, int64_t ld_g,
                                              int32_t B, double* w_out, int32_t device, void* stream, char* errbuf,
                                              int32_t errbuf_len) {
    char msg[256];
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    if (!phi || !g || !w_out) { say(errbuf, errbuf_len, "admm_phit_apply_static: phi, g and w_out must be non-null device pointers"); return ADMM_EINVAL; }
    if (N < 1 || n < 1 || B < 1 || ld < n || ld_g < N) {
        say(errbuf, errbuf_len, "admm_phit_apply_static: need N >= 1, n >= 1, B >= 1, ld >= n, ld_g >= N"); return ADMM_EINVAL;
    }
    const int64_t tiles_m = (n + kTile - 1) / kTile, tiles_q = ((int64_t)B + kTile - 1) / kTile;
    if ((int64_t)B * n > kPartialFloats || tiles_m * tiles_q > kTicketWords || tiles_q > 65535) {
        std::snprintf(msg, sizeof msg, "admm_phit_apply_static: B * n = %lld exceeds the static scratch (at most %lld outputs, %lld "
                      "output tiles of 64 x 64; ADMM_STATIC_SCRATCH_BYTES = %lld): use admm_setup / admm_contract_probe instead",
                      (long long)((int64_t)B * n), (long long)kPartialFloats, (long long)kTicketWords, (long long)ADMM_STATIC_SCRATCH_BYTES);
        say(errbuf, errbuf_len, msg); return ADMM_EINVAL;
    }
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count < 1) { cudaGetLastError(); say(errbuf, errbuf_len, "admm_phit_apply_static: no CUDA device"); return ADMM_ECUDA; }
    if (device < 0 || device >= count || device >= kMaxDevices) { say(errbuf, errbuf_len, "admm_phit_apply_static: device ordinal out of range"); return ADMM_EINVAL; }
    DeviceGuard guard;
    cudaError_t e = cudaGetDevice(&guard.prev);
    if (e == cudaSuccess && guard.prev != device) { e = cudaSetDevice(device); guard.switched = (e == cudaSuccess); }
    if (e != cudaSuccess) {
        std::snprintf(msg, sizeof msg, "admm_phit_apply_static: cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
        cudaGetLastError(); say(errbuf, errbuf_len, msg); return ADMM_ECUDA;
    }
    DeviceSlot slot;
    {   // set-up, once per device, with that device current: the device address of the scratch array
        std::lock_guard<std::mutex> lock(g_mu);
        DeviceSlot& s = g_slot[device];
        if (!s.ready) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e == cudaSuccess) e = cudaDeviceGetAttribute(&s.sm_count, cudaDevAttrMultiProcessorCount, device);
            if (e != cudaSuccess || !p) {
                std::snprintf(msg, sizeof msg, "admm_phit_apply_static: cudaGetSymbolAddress on device %d: %s (the library is built for sm_100a only)",
                              device, cudaGetErrorString(e));
                cudaGetLastError(); say(errbuf, errbuf_len, msg); return ADMM_ECUDA;
            }
            s.scratch = static_cast<unsigned char*>(p);
            s.ready = true;
        }
        slot = s;
    }
    if (!on_device(phi, device) || !on_device(g, device) || !on_device(w_out, device)) {
        say(errbuf, errbuf_len, "admm_phit_apply_static: phi, g and w_out must point to memory of the given device"); return ADMM_EINVAL;
    }
    // splits: enough blocks for two waves, each split at least 256 points deep, partial sums within the scratch
    const int64_t tiles = tiles_m * tiles_q;
    int64_t splits = (2 * (int64_t)slot.sm_count + tiles - 1) / tiles;
    splits = std::min<int64_t>(splits, (N + 255) / 256);
    splits = std::min<int64_t>(splits, kPartialFloats / ((int64_t)B * n));
    splits = std::max<int64_t>(1, std::min<int64_t>(splits, kMaxSplits));
    const int64_t k_per_split = ((N + splits - 1) / splits + kKStep - 1) / kKStep * kKStep;
    splits = (N + k_per_split - 1) / k_per_split;                        // no empty split: every block of a tile takes a ticket
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // the arrival counters must start at zero (they do after a completed call; a call that was aborted may have left some behind)
    e = cudaMemsetAsync(slot.scratch, 0, (size_t)tiles * sizeof(unsigned int), st);
    if (e == cudaSuccess) {
        dim3 grid((unsigned)tiles_m, (unsigned)tiles_q, (unsigned)splits);
        phit_apply_static_kernel<<<grid, 256, 0, st>>>(phi, N, n, ld, g, (int)B, ld_g, k_per_split, slot.scratch, w_out);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        std::snprintf(msg, sizeof msg, "admm_phit_apply_static: launch failed: %s", cudaGetErrorString(e));
        say(errbuf, errbuf_len, msg); return ADMM_ECUDA;
    }
    return ADMM_OK;
}
