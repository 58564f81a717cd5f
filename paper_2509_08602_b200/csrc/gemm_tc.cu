// The two dose-rate contractions of one ADMM iteration as tcgen05 kernels (sm_100a).
//
//   K1  W   = Phi^T . G      "A r1"   of Eq. (6), PAPER.md:89   big operand PhiT [n][N], small operand G  [B][N]
//   K3  Q   = Phi   . V      "A^T v"  of Eq. (7), PAPER.md:93   big operand Phi  [N][n], small operand V  [B][n]
//   OBJ dose= Phi   . T      primal objective, PAPER.md:183     (K3's mainloop, another epilogue)
//
// One kernel serves all three.  D[128 rows of the big operand][plans] accumulates in TMEM (fp32).
// Both operands are K-major fp32 tiles of 32 elements (one 128-byte swizzle row) staged by TMA.
// "fp32 path" = 3xTF32: the small operand arrives pre-split (hi on the tf32 grid, lo = x - hi, both written
// by the producing epilogue); the big operand (Phi) is read ONCE from HBM as fp32 and split on chip by four
// converter warps (hi = bits above the tf32 cut, lo = x - hi, exact), then
//     D += Phi_lo.G_hi ; D += Phi_hi.G_lo ; D += Phi_hi.G_hi          (small terms first)
// With mma_passes == 2 the big operand is already on the tf32 grid (ADMM_STORAGE_FP32_TF32), no converter.
//
// Warp roles (320 threads, 1 CTA / SM, persistent over a host-built unit list):
//   warp 0      TMA producer (one lane)           warp 1      UMMA issuer (one lane) + TMEM alloc/dealloc
//   warps 2-5   converter (hi/lo split in smem)    warps 6-9   epilogue (TMEM -> registers -> global)
// Pipelines: smem ring full[s] -> (conv[s]) -> empty[s]; TMEM double buffer tmem_full[a] / tmem_empty[a].
#include <cstdio>
#include <cstring>
#include "admm_internal.h"
#include "epilogue.cuh"
#include "tc_ptx.cuh"

namespace {

constexpr int kTileBytes = kTileM * kBlockK * 4;       // 16 KB: 128 rows x 128 B
constexpr int kBoxBytes = kBoxRows * kBlockK * 4;      // 4 KB
constexpr int kMaxStages = 8;
constexpr int kAccCols = 256;                          // TMEM columns per accumulator stage (DRAIN = false)
constexpr int kDrainCols = 128;                        // DRAIN: 2 main + 2 correction accumulators of 128 columns
constexpr int kSmemLimit = 227 * 1024;

struct Ctrl {
    uint64_t full[kMaxStages];
    uint64_t conv[kMaxStages];
    uint64_t empty[kMaxStages];
    uint64_t tmem_full[2];
    uint64_t tmem_empty[2];
    uint64_t small_full[2];     // DRAIN: accumulator of the correction terms, one per unit
    uint64_t small_empty[2];
    uint32_t tmem_base;
    uint32_t pad;
};

__host__ __device__ inline int stage_bytes(int mma_passes, int n_mma) {
    return kTileBytes * (mma_passes == 3 ? 2 : 1) + 2 * n_mma * kBlockK * 4;
}
__host__ __device__ inline int acc_bytes(int n_mma) { return 8 * n_mma * 8 * 4; }   // [8 warps][n_mma][8] floats

// Everything one epilogue thread needs to process columns (plans) of its row.
struct EpiCtx {
    bool valid; int lrow; int64_t row; int cls; float a_k, sense, thr; bool resid; int64_t mword; int lane;
    float* wacc; int slot;
};

// 16 consecutive columns c0..c0+15 of this thread's row: q[jj] = accumulator of plan (slot0 + c0 + jj).
__device__ __forceinline__ void epi_cols16(const TcLaunch& L, const EpiCtx& cx, int c0, const float* q) {
    const EpiParams& ep = L.ep;
    const int n_act = ep.n_slots_active;
    if (L.epi == EPI_K1_PARTIAL) {
        float* dst = ep.partial + ((int64_t)cx.slot * ep.n_mma) * kTileM + cx.lrow;
#pragma unroll
        for (int jj = 0; jj < 16; ++jj)
            if (c0 + jj < n_act) dst[(int64_t)(c0 + jj) * kTileM] = q[jj];
        return;
    }
    if (L.epi == EPI_RAW) {
#pragma unroll
        for (int jj = 0; jj < 16; ++jj)
            if (c0 + jj < n_act && cx.valid) ep.qraw[(int64_t)(ep.slot0 + c0 + jj) * ep.ldN + cx.row] = q[jj];
        return;
    }
    float so[16];
    uint32_t mw[16];
    if (cx.valid) {
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) {
            const int p = c0 + jj;
            so[jj] = 0.0f; mw[jj] = 0xFFFFFFFFu;
            if (p < n_act) {
                if (L.epi == EPI_K3_STATE) so[jj] = ep.s1[(int64_t)(ep.slot0 + p) * ep.ldN + cx.row];
                if (ep.mask) mw[jj] = __ldg(ep.mask + (int64_t)__ldg(ep.slot_plan + ep.slot0 + p) * ep.mask_words + cx.mword);
            }
        }
    }
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) {
        const int p = c0 + jj;
        if (p >= n_act) break;                      // warp-uniform
        float racc[kNumResid] = {0.f, 0.f, 0.f, 0.f, 0.f};
        float hinge = 0.f;
        if (cx.valid) {
            const bool on = (mw[jj] >> (cx.row & 31)) & 1u;
            if (L.epi == EPI_K3_STATE) {
                const float ub = on ? __ldg(ep.utab + cx.cls * kMaxBpad + ep.slot0 + p) : 0.0f;
                const float cr = __ldg(ep.crtab + cx.cls * kMaxBpad + ep.slot0 + p);
                Epi1Out o = epi1_element(so[jj], q[jj], cx.a_k, cr, ub, cx.resid, racc);
                const int64_t idx = (int64_t)(ep.slot0 + p) * ep.ldN + cx.row;
                ep.s1[idx] = o.s_new;
                ep.g_hi[idx] = o.g_hi;
                ep.g_lo[idx] = o.g_lo;
            } else {
                hinge = on ? fmaxf(0.0f, cx.sense * (cx.thr - q[jj])) : 0.0f;
            }
        }
        if (cx.resid) {
#pragma unroll
            for (int t = 0; t < kNumResid; ++t) {
                float v = warp_sum(racc[t]);
                if (cx.lane == 0) cx.wacc[p * 8 + t] += v;
            }
        } else if (L.epi == EPI_OBJECTIVE) {
            for (int k = 0; k < kMaxClasses; ++k) {
                float v = warp_sum((cx.valid && cx.cls == k) ? hinge : 0.0f);
                if (cx.lane == 0) cx.wacc[p * 8 + k] += v;
            }
        }
    }
}

// DRAIN = true  (fp32 path): the TMEM accumulator is emptied every L.chunk_kb k-blocks into fp32 register
//   master sums by 8 epilogue warps (two per TMEM lane group, half of the columns each).  tcgen05.mma
//   accumulates with round-toward-zero (measured: bias -2^-25 per MMA, linear in K, coherent over
//   iterations); summing short chunks with round-to-nearest FADDs removes that bias.  n_mma <= 128.
// DRAIN = false: one chunk per unit, 4 epilogue warps read the finished accumulator once.  n_mma <= 256.
template <bool DRAIN>
__global__ void __launch_bounds__(DRAIN ? 448 : 320, 1) admm_contract_kernel(const __grid_constant__ TcLaunch L) {
    constexpr int kThreads = DRAIN ? 448 : 320;
    constexpr int kEpiWarps = DRAIN ? 8 : 4;
    extern __shared__ __align__(1024) uint8_t smem[];
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int n_mma = L.ep.n_mma;
    const int passes = L.mma_passes;
    const int sbytes = stage_bytes(passes, n_mma);
    // carve: [stages x stage][acc][ctrl]
    int n_stages = (kSmemLimit - 1024 - (int)sizeof(Ctrl) - acc_bytes(n_mma)) / sbytes;
    if (n_stages > kMaxStages) n_stages = kMaxStages;
    uint8_t* stage_base = smem;
    float* acc = reinterpret_cast<float*>(smem + n_stages * sbytes);
    Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem + n_stages * sbytes + acc_bytes(n_mma));

    const int unit_begin = L.cta_unit_begin[blockIdx.x];
    const int unit_end = L.cta_unit_begin[blockIdx.x + 1];
    const int chunk_kb = L.chunk_kb;

    if (threadIdx.x == 0) {
        for (int s = 0; s < n_stages; ++s) {
            tc::mbar_init(&ctrl->full[s], 1);
            tc::mbar_init(&ctrl->conv[s], 128);
            tc::mbar_init(&ctrl->empty[s], 1);
        }
        for (int a = 0; a < 2; ++a) {
            tc::mbar_init(&ctrl->tmem_full[a], 1);
            tc::mbar_init(&ctrl->tmem_empty[a], kEpiWarps * 32);
            tc::mbar_init(&ctrl->small_full[a], 1);
            tc::mbar_init(&ctrl->small_empty[a], kEpiWarps * 32);
        }
        tc::fence_barrier_init();
        tc::tma_prefetch_desc(&L.map_big);
        tc::tma_prefetch_desc(&L.map_small_hi);
        tc::tma_prefetch_desc(&L.map_small_lo);
    }
    for (int i = threadIdx.x; i < acc_bytes(n_mma) / 4; i += kThreads) acc[i] = 0.0f;
    if (warp == 1) tc::tmem_alloc(&ctrl->tmem_base, 512);
    tc::tcgen05_fence_before();
    __syncthreads();
    tc::tcgen05_fence_after();
    const uint32_t tmem_base = ctrl->tmem_base;

    auto stage_a_raw = [&](int s) { return stage_base + s * sbytes; };
    auto stage_a_lo = [&](int s) { return stage_base + s * sbytes + kTileBytes; };
    auto stage_b_hi = [&](int s) { return stage_base + s * sbytes + kTileBytes * (passes == 3 ? 2 : 1); };
    auto stage_b_lo = [&](int s) { return stage_b_hi(s) + n_mma * kBlockK * 4; };

    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer
        if (lane == 0) {
            int s = 0; uint32_t ph = 0;
            for (int u = unit_begin; u < unit_end; ++u) {
                const TcUnit un = L.units[u];
                const int nbox = (un.rows + kBoxRows - 1) / kBoxRows;
                const uint32_t bytes = nbox * kBoxBytes + 2 * n_mma * kBlockK * 4;
                for (int kb = 0; kb < un.kb_count; ++kb) {
                    tc::mbar_wait(&ctrl->empty[s], ph ^ 1);
                    tc::mbar_arrive_expect_tx(&ctrl->full[s], bytes);
                    const int k0 = (un.kb0 + kb) * kBlockK;
                    for (int b = 0; b < nbox; ++b)
                        tc::tma_load_2d(stage_a_raw(s) + b * kBoxBytes, &L.map_big, &ctrl->full[s], k0,
                                        un.row0 + b * kBoxRows, tc::kEvictFirst);
                    tc::tma_load_2d(stage_b_hi(s), &L.map_small_hi, &ctrl->full[s], k0, 0, tc::kEvictLast);
                    tc::tma_load_2d(stage_b_lo(s), &L.map_small_lo, &ctrl->full[s], k0, 0, tc::kEvictLast);
                    if (++s == n_stages) { s = 0; ph ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------ UMMA issuer
        if (lane == 0) {
            const uint32_t idesc = tc::umma_idesc(2u, kTileM, (uint32_t)n_mma);
            int s = 0; uint32_t ph = 0;
            int a = 0; uint32_t aph = 0;
            int b = 0; uint32_t bph = 0;
            for (int u = unit_begin; u < unit_end; ++u) {
                const TcUnit un = L.units[u];
                const int ck = DRAIN ? chunk_kb : un.kb_count;
                // DRAIN: correction terms (lo.hi + hi.lo) accumulate over the whole unit in their own accumulator
                const uint32_t d_small = tmem_base + 2 * kDrainCols + b * kDrainCols;
                if (DRAIN) {
                    tc::mbar_wait(&ctrl->small_empty[b], bph ^ 1);
                    tc::tcgen05_fence_after();
                }
                for (int kb0 = 0; kb0 < un.kb_count; kb0 += ck) {
                    const int nkb = min(ck, un.kb_count - kb0);
                    tc::mbar_wait(&ctrl->tmem_empty[a], aph ^ 1);
                    tc::tcgen05_fence_after();
                    const uint32_t d_tmem = tmem_base + a * (DRAIN ? kDrainCols : kAccCols);
                    for (int kb = 0; kb < nkb; ++kb) {
                        tc::mbar_wait(passes == 3 ? &ctrl->conv[s] : &ctrl->full[s], ph);
                        tc::tcgen05_fence_after();
                        const uint64_t a_raw = tc::umma_desc_k_sw128(tc::smem_u32(stage_a_raw(s)));
                        const uint64_t a_lo = tc::umma_desc_k_sw128(tc::smem_u32(stage_a_lo(s)));
                        const uint64_t b_hi = tc::umma_desc_k_sw128(tc::smem_u32(stage_b_hi(s)));
                        const uint64_t b_lo = tc::umma_desc_k_sw128(tc::smem_u32(stage_b_lo(s)));
#pragma unroll
                        for (int k = 0; k < kBlockK / 8; ++k) {
                            const uint64_t koff = (uint64_t)((k * 8 * 4) >> 4);   // 32 bytes per tf32 k-step
                            const uint32_t first = (kb | k) ? 1u : 0u;              // first MMA of this chunk
                            if (DRAIN) {
                                const uint32_t first_u = ((kb0 + kb) | k) ? 1u : 0u; // first MMA of this unit
                                if (passes == 3) {
                                    tc::umma_tf32(d_small, a_lo + koff, b_hi + koff, idesc, first_u);
                                    tc::umma_tf32(d_small, a_raw + koff, b_lo + koff, idesc, 1u);
                                } else {
                                    tc::umma_tf32(d_small, a_raw + koff, b_lo + koff, idesc, first_u);
                                }
                                tc::umma_tf32(d_tmem, a_raw + koff, b_hi + koff, idesc, first);
                            } else {
                                if (passes == 3) {
                                    tc::umma_tf32(d_tmem, a_lo + koff, b_hi + koff, idesc, first);
                                    tc::umma_tf32(d_tmem, a_raw + koff, b_lo + koff, idesc, 1u);
                                } else {
                                    tc::umma_tf32(d_tmem, a_raw + koff, b_lo + koff, idesc, first);
                                }
                                tc::umma_tf32(d_tmem, a_raw + koff, b_hi + koff, idesc, 1u);
                            }
                        }
                        tc::umma_commit(&ctrl->empty[s]);
                        if (++s == n_stages) { s = 0; ph ^= 1; }
                    }
                    tc::umma_commit(&ctrl->tmem_full[a]);
                    if (++a == 2) { a = 0; aph ^= 1; }
                }
                if (DRAIN) {
                    tc::umma_commit(&ctrl->small_full[b]);
                    if (++b == 2) { b = 0; bph ^= 1; }
                }
            }
        }
    } else if (warp < 6) {
        // ------------------------------------------------------------ converter: hi/lo split of the big operand
        if (passes == 3) {
            const int tid = threadIdx.x - 64;          // 0..127
            int s = 0; uint32_t ph = 0;
            for (int u = unit_begin; u < unit_end; ++u) {
                const TcUnit un = L.units[u];
                const int nvec = ((un.rows + kBoxRows - 1) / kBoxRows) * (kBoxBytes / 16);
                for (int kb = 0; kb < un.kb_count; ++kb) {
                    tc::mbar_wait(&ctrl->full[s], ph);
                    float4* raw = reinterpret_cast<float4*>(stage_a_raw(s));
                    float4* lo = reinterpret_cast<float4*>(stage_a_lo(s));
#pragma unroll 4
                    for (int i = tid; i < nvec; i += 128) {
                        float4 v = raw[i];
                        float4 hi, l;
                        hi.x = __uint_as_float(__float_as_uint(v.x) & 0xFFFFE000u); l.x = v.x - hi.x;
                        hi.y = __uint_as_float(__float_as_uint(v.y) & 0xFFFFE000u); l.y = v.y - hi.y;
                        hi.z = __uint_as_float(__float_as_uint(v.z) & 0xFFFFE000u); l.z = v.z - hi.z;
                        hi.w = __uint_as_float(__float_as_uint(v.w) & 0xFFFFE000u); l.w = v.w - hi.w;
                        raw[i] = hi;
                        lo[i] = l;
                    }
                    tc::fence_proxy_async_smem();
                    tc::mbar_arrive(&ctrl->conv[s]);
                    if (++s == n_stages) { s = 0; ph ^= 1; }
                }
            }
        }
    } else {
        // ------------------------------------------------------------ epilogue (one TMEM lane = one row per thread)
        const int ew = warp & 3;                       // TMEM lane group this warp may read
        const EpiParams& ep = L.ep;
        const int n16 = n_mma / 16;
        const int half = DRAIN ? ((warp - 6) >> 2) : 0;
        const int cbeg = DRAIN ? (half == 0 ? 0 : (n16 + 1) / 2) : 0;          // first 16-column group of this warp
        const int cend = DRAIN ? (half == 0 ? (n16 + 1) / 2 : n16) : n16;
        EpiCtx cx;
        cx.lane = lane;
        cx.wacc = acc + (warp - 6) * n_mma * 8;
        cx.resid = (L.epi == EPI_K3_STATE) && (ep.resid_partial != nullptr);
        int a = 0; uint32_t aph = 0;
        int b2 = 0; uint32_t bph2 = 0;
        for (int u = unit_begin; u < unit_end; ++u) {
            const TcUnit un = L.units[u];
            cx.lrow = ew * 32 + lane;
            cx.valid = cx.lrow < un.rows;
            cx.row = (int64_t)un.row0 + cx.lrow;
            cx.slot = un.slot;
            cx.cls = 0;
            if (cx.valid && L.epi != EPI_K1_PARTIAL && L.epi != EPI_RAW) cx.cls = ep.point_class[cx.row];
            cx.a_k = ep.a_cls[cx.cls]; cx.sense = ep.sense[cx.cls]; cx.thr = ep.thr[cx.cls];
            cx.mword = cx.row >> 5;
            const uint32_t lane_addr = tmem_base + ((uint32_t)(ew * 32) << 16);
            if (DRAIN) {
                float master[64];
#pragma unroll
                for (int i = 0; i < 64; ++i) master[i] = 0.0f;
                for (int kb0 = 0; kb0 < un.kb_count; kb0 += chunk_kb) {
                    tc::mbar_wait(&ctrl->tmem_full[a], aph);
                    tc::tcgen05_fence_after();
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) {
                        if (cbeg + cc < cend) {
                            uint32_t r[16];
                            tc::tmem_ld16(lane_addr + a * kDrainCols + (cbeg + cc) * 16, r);
                            tc::tmem_ld_wait(r);
#pragma unroll
                            for (int jj = 0; jj < 16; ++jj) master[cc * 16 + jj] += __uint_as_float(r[jj]);
                        }
                    }
                    tc::tcgen05_fence_before();
                    tc::mbar_arrive(&ctrl->tmem_empty[a]);
                    if (++a == 2) { a = 0; aph ^= 1; }
                }
                // the correction-term accumulator of this unit
                tc::mbar_wait(&ctrl->small_full[b2], bph2);
                tc::tcgen05_fence_after();
#pragma unroll
                for (int cc = 0; cc < 4; ++cc) {
                    if (cbeg + cc < cend) {
                        uint32_t r[16];
                        tc::tmem_ld16(lane_addr + 2 * kDrainCols + b2 * kDrainCols + (cbeg + cc) * 16, r);
                        tc::tmem_ld_wait(r);
#pragma unroll
                        for (int jj = 0; jj < 16; ++jj) master[cc * 16 + jj] += __uint_as_float(r[jj]);
                    }
                }
                tc::tcgen05_fence_before();
                tc::mbar_arrive(&ctrl->small_empty[b2]);
                if (++b2 == 2) { b2 = 0; bph2 ^= 1; }
#pragma unroll
                for (int cc = 0; cc < 4; ++cc)
                    if (cbeg + cc < cend) epi_cols16(L, cx, (cbeg + cc) * 16, &master[cc * 16]);
            } else {
                tc::mbar_wait(&ctrl->tmem_full[a], aph);
                tc::tcgen05_fence_after();
                for (int c = cbeg; c < cend; ++c) {
                    uint32_t r[16];
                    tc::tmem_ld16(lane_addr + a * kAccCols + c * 16, r);
                    tc::tmem_ld_wait(r);
                    float q[16];
#pragma unroll
                    for (int jj = 0; jj < 16; ++jj) q[jj] = __uint_as_float(r[jj]);
                    epi_cols16(L, cx, c * 16, q);
                }
                tc::tcgen05_fence_before();
                tc::mbar_arrive(&ctrl->tmem_empty[a]);
                if (++a == 2) { a = 0; aph ^= 1; }
            }
        }
    }

    __syncthreads();
    // per-CTA partial sums -> global (fixed order over the epilogue warps), deterministic
    if (L.epi == EPI_K3_STATE && L.ep.resid_partial != nullptr) {
        for (int i = threadIdx.x; i < L.ep.n_slots_active * kNumResid; i += kThreads) {
            const int p = i / kNumResid, t = i % kNumResid;
            float v = 0.f;
            for (int w = 0; w < kEpiWarps; ++w) v += acc[(w * n_mma + p) * 8 + t];
            L.ep.resid_partial[((int64_t)blockIdx.x * kMaxBpad + L.ep.slot0 + p) * kNumResid + t] = v;
        }
    } else if (L.epi == EPI_OBJECTIVE) {
        for (int i = threadIdx.x; i < L.ep.n_slots_active * kMaxClasses; i += kThreads) {
            const int p = i / kMaxClasses, k = i % kMaxClasses;
            double v = 0.0;
            for (int w = 0; w < kEpiWarps; ++w) v += (double)acc[(w * n_mma + p) * 8 + k];
            L.ep.hinge_partial[((int64_t)blockIdx.x * kMaxBpad + L.ep.slot0 + p) * kMaxClasses + k] = v;
        }
    }
    if (warp == 1) {
        tc::tcgen05_fence_after();
        tc::tmem_dealloc(tmem_base, 512);
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

}  // namespace

admm_status tc_init(admm_handle* h) {
    if (!g_encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
            h->err = "cuTensorMapEncodeTiled not available from the driver";
            return ADMM_ECUDA;
        }
        g_encode = reinterpret_cast<EncodeTiledFn>(fn);
    }
    cudaError_t e = cudaFuncSetAttribute(admm_contract_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(admm_contract_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
    if (e != cudaSuccess) {
        h->err = std::string("cudaFuncSetAttribute(max dynamic smem): ") + cudaGetErrorString(e);
        return ADMM_ECUDA;
    }
    return ADMM_OK;
}

// 2-D fp32 tensor [rows][cols] with row stride ld_elems, box = {32 cols (128 B), box_rows}, 128-byte swizzle,
// out-of-bounds elements read as zero.
admm_status tc_make_map(admm_handle* h, CUtensorMap* out, const void* base, int64_t rows, int64_t cols,
                        int64_t ld_elems, int box_rows) {
    cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t gstride[1] = {(cuuint64_t)ld_elems * 4};
    cuuint32_t box[2] = {(cuuint32_t)kBlockK, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char buf[160];
        snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (%d) rows=%lld cols=%lld ld=%lld box_rows=%d", (int)r,
                 (long long)rows, (long long)cols, (long long)ld_elems, box_rows);
        h->err = buf;
        return ADMM_ECUDA;
    }
    return ADMM_OK;
}

admm_status tc_launch(admm_handle* h, const TcLaunch& L) {
    const int n_mma = L.ep.n_mma;
    if (n_mma < 16 || n_mma > kMaxMmaN || (n_mma % 16) != 0) {
        h->err = "tc_launch: n_mma must be a multiple of 16 in [16, 256]";
        return ADMM_EINVAL;
    }
    const int sbytes = stage_bytes(L.mma_passes, n_mma);
    int n_stages = (kSmemLimit - 1024 - (int)sizeof(Ctrl) - acc_bytes(n_mma)) / sbytes;
    if (n_stages < 2) {
        h->err = "tc_launch: fewer than 2 pipeline stages fit in shared memory";
        return ADMM_EINVAL;
    }
    if (L.chunk_kb > 0) {
        if (n_mma > 128) { h->err = "tc_launch: the drained (fp32) path needs n_mma <= 128"; return ADMM_EINVAL; }
        admm_contract_kernel<true><<<L.grid, 448, kSmemLimit, h->stream>>>(L);
    } else {
        admm_contract_kernel<false><<<L.grid, 320, kSmemLimit, h->stream>>>(L);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        h->err = std::string("admm_contract_kernel launch: ") + cudaGetErrorString(e);
        return ADMM_ECUDA;
    }
    h->launch_count++;
    return ADMM_OK;
}
