// The two dose-rate contractions of one ADMM iteration as tcgen05 kernels (sm_100a).
//
//   K1  W   = Phi^T . G      "A r1"   of Eq. (6), PAPER.md:89   big operand PhiT [n][N], small operand G  [B][N]
//   K3  Q   = Phi   . V      "A^T v"  of Eq. (7), PAPER.md:93   big operand Phi  [N][n], small operand V  [B][n]
//   OBJ dose= Phi   . T      primal objective, PAPER.md:183     (K3's mainloop, another epilogue)
//
// D[128 rows of the big operand][plans] accumulates in TMEM (fp32).  Both operands are K-major tiles of 128-byte rows
// (32 fp32 / 64 bf16 elements, one swizzle row) staged by TMA; the big operand is stored tile-major in HBM.
// "fp32 path" = 3xTF32: the small operand arrives pre-split (hi on the tf32 grid, lo = x - hi, both written by the producing
// epilogue); the big operand (Phi) is read ONCE from HBM as fp32 and split on chip.
//
// Three kernels, chosen by tc_launch():
//   admm_contract_f32_kernel   passes of <= 96 plans, every storage mode (3xTF32: converter -> TMEM A ring, TS-form MMAs,
//                              drained accumulation, staged epilogue; tf32 / bf16 storage: A straight from shared memory)
//   admm_contract_wide_kernel  3xTF32 passes of 97..224 plans: hi/lo tiles in shared memory, SS-form MMAs, drained
//                              accumulation, epilogue from the drain warps' registers
//   admm_contract_kernel       tf32 / bf16 storage, passes of 97..256 plans: undrained accumulation, epilogue from TMEM
#include <cstdio>
#include <cstring>
#include "admm_internal.h"
#include "epilogue.cuh"
#include "tc_ptx.cuh"

namespace {

constexpr int kTileBytes = kTileM * kBlockK * 4;       // 16 KB: 128 rows x 128 B
constexpr int kBoxBytes = kBoxRows * kBlockK * 4;      // 4 KB
constexpr int kMaxStages = 8;
constexpr int kAccCols = 256;                          // TMEM columns per accumulator stage of admm_contract_kernel
constexpr int kSmemLimit = 227 * 1024;

struct Ctrl {
    uint64_t full[kMaxStages];
    uint64_t empty[kMaxStages];
    uint64_t tmem_full[2];
    uint64_t tmem_empty[2];
    uint32_t tmem_base;
    uint32_t pad;
};

__host__ __device__ inline int stage_bytes(int n_mma) { return kTileBytes + 2 * n_mma * kBlockK * 4; }
__host__ __device__ inline int acc_bytes(int n_mma) { return 4 * n_mma * 8 * 4; }   // [4 warps][n_mma][8] floats

// Everything one epilogue thread needs to process columns (plans) of its row.
struct EpiCtx {
    bool valid; int lrow; int64_t row; int cls; float a_k, sense, thr; bool resid; int64_t mword; int lane;
    float* wacc; int slot; int n_act;
};

// 16 consecutive columns c0..c0+15 of this thread's row: q[jj] = accumulator of plan (slot0 + c0 + jj).
// Inlined, arrays in registers, the 16 state loads of the group in flight together (unconditional, indices clamped; only
// the stores are predicated) -- see epilogue_unit_t for why.
__device__ __forceinline__ void epi_cols16(const TcLaunch& L, const EpiCtx& cx, int c0, const float (&q)[16]) {
    const EpiParams& ep = L.ep;
    const int n_act = cx.n_act;
    const int epi = L.epi;
    if (epi == EPI_K1_PARTIAL) {
        float* dst = ep.partial + ((int64_t)cx.slot * ep.n_mma) * kTileM + cx.lrow;
#pragma unroll
        for (int jj = 0; jj < 16; ++jj)
            if (c0 + jj < n_act) dst[(int64_t)(c0 + jj) * kTileM] = q[jj];
        return;
    }
    if (epi == EPI_RAW) {
#pragma unroll
        for (int jj = 0; jj < 16; ++jj)
            if (c0 + jj < n_act && cx.valid) ep.qraw[(int64_t)(ep.slot0 + c0 + jj) * ep.ldN + cx.row] = q[jj];
        return;
    }
    if (c0 >= n_act) return;                                         // warp-uniform
    const int p_last = n_act - 1;
    const bool has_mask = ep.mask != nullptr;
    const uint32_t* mrow = has_mask ? ep.mask + cx.mword : reinterpret_cast<const uint32_t*>(ep.slot_plan);
    const float* s1c = ep.s1 + (int64_t)ep.slot0 * ep.ldN + cx.row;     // cx.row is clamped to a row that exists
    const bool bf16 = ep.small_bf16 != 0;
    float so[16];
    uint32_t mw[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) {
        const int p = min(c0 + jj, p_last);
        so[jj] = (epi == EPI_K3_STATE) ? s1c[(int64_t)p * ep.ldN] : 0.0f;
        mw[jj] = has_mask ? __ldg(mrow + (int64_t)__ldg(ep.slot_plan + ep.slot0 + p) * ep.mask_words) : 0xFFFFFFFFu;
    }
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) {
        const int p = min(c0 + jj, p_last);
        const bool inb = c0 + jj < n_act;                            // warp-uniform
        const bool live = cx.valid && inb;
        const bool on = (mw[jj] >> (cx.row & 31)) & 1u;
        float racc[kNumResid] = {0.f, 0.f, 0.f, 0.f, 0.f};
        float hinge = 0.f;
        if (epi == EPI_K3_STATE) {
            float rtmp[kNumResid] = {0.f, 0.f, 0.f, 0.f, 0.f};
            const float ub = on ? __ldg(ep.utab + cx.cls * kMaxBpad + ep.slot0 + p) : 0.0f;
            const float cr = __ldg(ep.crtab + cx.cls * kMaxBpad + ep.slot0 + p);
            Epi1Out o = epi1_element(so[jj], q[jj], cx.a_k, cr, ub, cx.resid, rtmp);
            if (live) {
                ep.s1[(int64_t)(ep.slot0 + p) * ep.ldN + cx.row] = o.s_new;
                emit_small(ep.g_hi, ep.g_lo, (int64_t)(ep.slot0 + p) * ep.ldN, cx.row, o.g, bf16);
#pragma unroll
                for (int t = 0; t < kNumResid; ++t) racc[t] = rtmp[t];
            }
        } else {
            hinge = (live && on) ? fmaxf(0.0f, cx.sense * (cx.thr - q[jj])) : 0.0f;
        }
        if (!inb) continue;
        if (cx.resid) {
#pragma unroll
            for (int t = 0; t < kNumResid; ++t) {
                float v = warp_sum(racc[t]);
                if (cx.lane == 0) cx.wacc[p * 8 + t] += v;
            }
        } else if (epi == EPI_OBJECTIVE) {
#pragma unroll 1
            for (int k = 0; k < kMaxClasses; ++k) {
                float v = warp_sum((live && cx.cls == k) ? hinge : 0.0f);
                if (cx.lane == 0) cx.wacc[p * 8 + k] += v;
            }
        }
    }
}

// tf32 / bf16 storage, passes of 97..256 plans (B = 441 in two passes).  The big operand is exact in the operand format, so the
// A tile goes straight from shared memory into the MMAs; the plan operand is a hi/lo pair: two MMAs per 32-byte k-step into ONE
// accumulator (lo first).  One accumulation per unit (no drain: the reduced-storage modes have a 1e-2 budget), two TMEM accumulator
// stages of 256 columns so the 4 epilogue warps read tile i while the MMAs of tile i+1 run.
// Warp roles (320 threads, 1 CTA / SM, persistent over a host-built unit list):
//   warp 0  TMA producer (one lane)      warp 1  UMMA issuer (one lane) + TMEM alloc/dealloc      warps 6-9  epilogue
__global__ void __launch_bounds__(320, 1) admm_contract_kernel(const __grid_constant__ TcLaunch L) {
    constexpr int kThreads = 320;
    constexpr int kEpiWarps = 4;
    extern __shared__ __align__(1024) uint8_t smem[];
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int n_mma = L.ep.n_mma;
    const int n_act = eff_nact(L.ep);
    if (n_act <= 0) return;                               // the whole pass froze since the host sized this launch
    const int sbytes = stage_bytes(n_mma);
    // carve: [stages x stage][acc][ctrl]
    int n_stages = (kSmemLimit - 1024 - (int)sizeof(Ctrl) - acc_bytes(n_mma)) / sbytes;
    if (n_stages > kMaxStages) n_stages = kMaxStages;
    uint8_t* stage_base = smem;
    float* acc = reinterpret_cast<float*>(smem + n_stages * sbytes);
    Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem + n_stages * sbytes + acc_bytes(n_mma));

    const int unit_begin = L.cta_unit_begin[blockIdx.x];
    const int unit_end = L.cta_unit_begin[blockIdx.x + 1];

    if (threadIdx.x == 0) {
        for (int s = 0; s < n_stages; ++s) {
            tc::mbar_init(&ctrl->full[s], 1);
            tc::mbar_init(&ctrl->empty[s], 1);
        }
        for (int a = 0; a < 2; ++a) {
            tc::mbar_init(&ctrl->tmem_full[a], 1);
            tc::mbar_init(&ctrl->tmem_empty[a], kEpiWarps * 32);
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

    auto stage_a = [&](int s) { return stage_base + s * sbytes; };
    auto stage_b_hi = [&](int s) { return stage_base + s * sbytes + kTileBytes; };
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
                    const int k0 = (un.kb0 + kb) * L.kblk;
                    const int trow = ((un.row0 >> 7) * L.big_kb_total + un.kb0 + kb) * kTileM;     // tile-major big operand
                    for (int b = 0; b < nbox; ++b)
                        tc::tma_load_2d(stage_a(s) + b * kBoxBytes, &L.map_big, &ctrl->full[s], 0,
                                        trow + b * kBoxRows, tc::kEvictFirst);
                    tc::tma_load_2d(stage_b_hi(s), &L.map_small_hi, &ctrl->full[s], k0, 0, tc::kEvictLast);
                    tc::tma_load_2d(stage_b_lo(s), &L.map_small_lo, &ctrl->full[s], k0, 0, tc::kEvictLast);
                    if (++s == n_stages) { s = 0; ph ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------ UMMA issuer
        if (lane == 0) {
            const bool bf16 = L.mma_kind == 1;
            const uint32_t idesc = tc::umma_idesc(bf16 ? 1u : 2u, kTileM, (uint32_t)n_mma);
            int s = 0; uint32_t ph = 0;
            int a = 0; uint32_t aph = 0;
            for (int u = unit_begin; u < unit_end; ++u) {
                const TcUnit un = L.units[u];
                tc::mbar_wait(&ctrl->tmem_empty[a], aph ^ 1);
                tc::tcgen05_fence_after();
                const uint32_t d_tmem = tmem_base + a * kAccCols;
                for (int kb = 0; kb < un.kb_count; ++kb) {
                    tc::mbar_wait(&ctrl->full[s], ph);
                    tc::tcgen05_fence_after();
                    const uint64_t a_desc = tc::umma_desc_k_sw128(tc::smem_u32(stage_a(s)));
                    const uint64_t b_hi = tc::umma_desc_k_sw128(tc::smem_u32(stage_b_hi(s)));
                    const uint64_t b_lo = tc::umma_desc_k_sw128(tc::smem_u32(stage_b_lo(s)));
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const uint64_t koff = (uint64_t)(2 * k);                // 32 bytes per k-step (8 tf32 / 16 bf16 elements)
                        const uint32_t first = (kb | k) ? 1u : 0u;              // first MMA of this unit overwrites
                        if (bf16) {
                            tc::umma_f16(d_tmem, a_desc + koff, b_lo + koff, idesc, first);
                            tc::umma_f16(d_tmem, a_desc + koff, b_hi + koff, idesc, 1u);
                        } else {
                            tc::umma_tf32(d_tmem, a_desc + koff, b_lo + koff, idesc, first);
                            tc::umma_tf32(d_tmem, a_desc + koff, b_hi + koff, idesc, 1u);
                        }
                    }
                    tc::umma_commit(&ctrl->empty[s]);
                    if (++s == n_stages) { s = 0; ph ^= 1; }
                }
                tc::umma_commit(&ctrl->tmem_full[a]);
                if (++a == 2) { a = 0; aph ^= 1; }
            }
        }
    } else if (warp >= 6) {
        // ------------------------------------------------------------ epilogue (one TMEM lane = one row per thread)
        const int ew = warp & 3;                       // TMEM lane group this warp may read
        const EpiParams& ep = L.ep;
        const int n16 = n_mma / 16;
        EpiCtx cx;
        cx.lane = lane;
        cx.n_act = n_act;
        cx.wacc = acc + (warp - 6) * n_mma * 8;
        cx.resid = (L.epi == EPI_K3_STATE) && (ep.resid_partial != nullptr);
        int a = 0; uint32_t aph = 0;
        for (int u = unit_begin; u < unit_end; ++u) {
            const TcUnit un = L.units[u];
            cx.lrow = ew * 32 + lane;
            cx.valid = cx.lrow < un.rows;
            cx.row = (int64_t)un.row0 + (cx.valid ? cx.lrow : 0);     // idle lanes load from a row that exists
            cx.slot = un.slot;
            cx.cls = 0;
            if (cx.valid && L.epi != EPI_K1_PARTIAL && L.epi != EPI_RAW) cx.cls = ep.point_class[cx.row];
            cx.a_k = ep.a_cls[cx.cls]; cx.sense = ep.sense[cx.cls]; cx.thr = ep.thr[cx.cls];
            cx.mword = cx.row >> 5;
            const uint32_t lane_addr = tmem_base + ((uint32_t)(ew * 32) << 16);
            tc::mbar_wait(&ctrl->tmem_full[a], aph);
            tc::tcgen05_fence_after();
            for (int c = 0; c < n16; ++c) {
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

    __syncthreads();
    // per-CTA partial sums -> global (fixed order over the epilogue warps), deterministic
    if (L.epi == EPI_K3_STATE && L.ep.resid_partial != nullptr) {
        for (int i = threadIdx.x; i < n_act * kNumResid; i += kThreads) {
            const int p = i / kNumResid, t = i % kNumResid;
            float v = 0.f;
            for (int w = 0; w < kEpiWarps; ++w) v += acc[(w * n_mma + p) * 8 + t];
            L.ep.resid_partial[((int64_t)blockIdx.x * kMaxBpad + L.ep.slot0 + p) * kNumResid + t] = v;
        }
    } else if (L.epi == EPI_OBJECTIVE) {
        for (int i = threadIdx.x; i < n_act * kMaxClasses; i += kThreads) {
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


// Epilogue of one unit from a staged accumulator tile qs[col][128 rows] in shared memory (written by the drain warps).
// One warp = 32 consecutive rows (lane = row), a loop over the plans in batches of 16 whose s1 loads are all in flight
// together; it runs concurrently with the MMAs / drains of the next unit.  Specialised at compile time on the epilogue
// kind and on whether residual sums are wanted: the hot instance (K3, no residuals) is ~40 instructions per plan (an
// earlier all-in-one version was instruction-fetch bound).  wacc: this warp's [n_mma][8] partial sums.
// Pull the s1 tile of a unit into L2 long before its epilogue needs it (the epilogue warps are otherwise exposed to
// the loaded HBM latency once per batch of plans).
__device__ __forceinline__ void prefetch_s1_tile(const TcLaunch& L, const TcUnit& un, int wq, int lane, int p_begin, int p_end) {
    const EpiParams& ep = L.ep;
    const int lrow = wq * 32 + lane;
    if (L.epi != EPI_K3_STATE || lrow >= un.rows) return;
    const float* s1p = ep.s1 + (int64_t)ep.slot0 * ep.ldN + un.row0 + lrow;
    for (int p = p_begin; p < p_end; ++p)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(s1p + (int64_t)p * ep.ldN));
}

// Epilogue of one unit from a staged accumulator tile qs[col][128 rows] in shared memory (written by the drain warps).
// One warp = 32 consecutive rows (lane = row) x the plans [p_begin, p_end), in batches of 8 whose loads are all in
// flight together; it runs concurrently with the MMAs / drains of the next unit.  Specialised at compile time on the
// epilogue kind and on whether residual sums are wanted, 32-bit element offsets: the hot instance (K3, no residuals,
// no mask) is ~35 instructions per plan.  Inlined on purpose: as a __noinline__ function it received the global-memory
// descriptor in ordinary registers and paid R2UR moves before EVERY load and store (measured with clock64: 23-30 us per
// unit, K3 was epilogue-bound: 134 us with bf16 storage against 78 us inlined).
// wacc: this warp's [n_mma][8] partial sums.
template <int EPI, bool RESID>
__device__ __forceinline__ void epilogue_unit_t(const TcLaunch& L, const TcUnit& un, const float* qs, int wq, int lane, float* wacc,
                                             int p_begin, int p_end) {
    const EpiParams& ep = L.ep;
    const int lrow = wq * 32 + lane;
    const bool valid = lrow < un.rows;
    const int64_t row = (int64_t)un.row0 + lrow;
    const float* qp = qs + lrow;
    if (EPI == EPI_K1_PARTIAL) {
        float* dst = ep.partial + ((int64_t)un.slot * ep.n_mma) * kTileM + lrow;
#pragma unroll 8
        for (int p = p_begin; p < p_end; ++p) dst[p * kTileM] = qp[p * kTileM];
        return;
    }
    if (EPI == EPI_RAW) {
        if (valid) {
            float* dst = ep.qraw + (int64_t)ep.slot0 * ep.ldN + row;
#pragma unroll 8
            for (int p = p_begin; p < p_end; ++p) dst[(int64_t)p * ep.ldN] = qp[p * kTileM];
        }
        return;
    }
    // Everything below is written so that the per-batch arrays stay in REGISTERS and the 8 global loads of a batch are in
    // flight together: loads are unconditional (indices clamped to a valid row / plan), only the stores are predicated.
    // (An earlier version guarded the loads with `if (live)` and left the unrolled loop with `break`: the arrays went to
    // local memory, every load was followed by a dependent STL, and the loads of a unit were served one DRAM latency at a
    // time -- 23-30 us per unit, measured with clock64, which made K3 epilogue-bound.)
    const int64_t rowc = valid ? row : (int64_t)un.row0;           // a row that exists, for the loads of idle lanes
    const int cls = ep.point_class[rowc];
    const float a_k = ep.a_cls[cls], sense = ep.sense[cls], thr = ep.thr[cls];
    const uint32_t mbit = (uint32_t)(rowc & 31);
    const float* utab = ep.utab + cls * kMaxBpad + ep.slot0;
    const float* crtab = ep.crtab + cls * kMaxBpad + ep.slot0;
    const int32_t* splan = ep.slot_plan + ep.slot0;
    const bool has_mask = ep.mask != nullptr;
    const uint32_t* mrow = has_mask ? ep.mask + (rowc >> 5) : reinterpret_cast<const uint32_t*>(ep.slot_plan);   // any valid address
    const uint32_t ldN = (uint32_t)ep.ldN;                     // Bpad * ldN < 2^32 (checked on the host)
    const int64_t base = (int64_t)ep.slot0 * ep.ldN + rowc;
    float* s1p = ep.s1 + base;
    float* ghp = reinterpret_cast<float*>(ep.g_hi) + base;       // fp32-container operands (tf32 grid)
    float* glp = reinterpret_cast<float*>(ep.g_lo) + base;
    const bool bf16 = ep.small_bf16 != 0;
    const int p_last = p_end - 1;
    constexpr int PB = 8;
    for (int p0 = p_begin; p0 < p_end; p0 += PB) {
        // phase 1: the long-latency loads (state, mask word) of the whole batch; the short ones (L1-resident tables,
        // shared memory) are taken in phase 2
        float so[PB];
        uint32_t mw[PB];
#pragma unroll
        for (int j = 0; j < PB; ++j) {
            const int p = min(p0 + j, p_last);
            so[j] = (EPI == EPI_K3_STATE) ? s1p[(uint32_t)p * ldN] : 0.0f;
            mw[j] = has_mask ? __ldg(mrow + (int64_t)__ldg(splan + p) * ep.mask_words) : 0xFFFFFFFFu;
        }
#pragma unroll
        for (int j = 0; j < PB; ++j) {
            const int p = min(p0 + j, p_last);
            const bool live = valid && (p0 + j < p_end);
            const bool on = (mw[j] >> mbit) & 1u;
            const float q = qp[p * kTileM];
            float racc[kNumResid] = {0.f, 0.f, 0.f, 0.f, 0.f};
            float hinge = 0.f;
            if (EPI == EPI_K3_STATE) {
                float rtmp[kNumResid] = {0.f, 0.f, 0.f, 0.f, 0.f};
                Epi1Out o = epi1_element(so[j], q, a_k, __ldg(crtab + p), on ? __ldg(utab + p) : 0.0f, RESID, rtmp);
                if (live) {
                    const uint32_t off = (uint32_t)p * ldN;
                    s1p[off] = o.s_new;
                    if (bf16) {
                        emit_small(ep.g_hi, ep.g_lo, (int64_t)(ep.slot0 + p) * ep.ldN, row, o.g, true);
                    } else {
                        const float ghi = tc::tf32_rna(o.g);
                        ghp[off] = ghi;
                        glp[off] = tc::tf32_rna(o.g - ghi);
                    }
#pragma unroll
                    for (int t = 0; t < kNumResid; ++t) racc[t] = rtmp[t];
                }
            } else {
                hinge = (live && on) ? fmaxf(0.0f, sense * (thr - q)) : 0.0f;
            }
            if (EPI == EPI_K3_STATE && RESID) {
                if (p0 + j < p_end) {                               // warp-uniform
#pragma unroll
                    for (int t = 0; t < kNumResid; ++t) {
                        float v = warp_sum(racc[t]);
                        if (lane == 0) wacc[p * 8 + t] += v;
                    }
                }
            } else if (EPI == EPI_OBJECTIVE) {
                if (p0 + j < p_end) {
#pragma unroll 1
                    for (int k = 0; k < kMaxClasses; ++k) {
                        float v = warp_sum((live && cls == k) ? hinge : 0.0f);
                        if (lane == 0) wacc[p * 8 + k] += v;
                    }
                }
            }
        }
    }
}

__device__ __forceinline__ void epilogue_unit(const TcLaunch& L, const TcUnit& un, const float* qs, int wq, int lane, float* wacc,
                                              int p_begin, int p_end) {
    switch (L.epi) {
        case EPI_K1_PARTIAL: epilogue_unit_t<EPI_K1_PARTIAL, false>(L, un, qs, wq, lane, wacc, p_begin, p_end); break;
        case EPI_K3_STATE:
            if (L.ep.resid_partial != nullptr) epilogue_unit_t<EPI_K3_STATE, true>(L, un, qs, wq, lane, wacc, p_begin, p_end);
            else epilogue_unit_t<EPI_K3_STATE, false>(L, un, qs, wq, lane, wacc, p_begin, p_end);
            break;
        case EPI_OBJECTIVE: epilogue_unit_t<EPI_OBJECTIVE, false>(L, un, qs, wq, lane, wacc, p_begin, p_end); break;
        default: epilogue_unit_t<EPI_RAW, false>(L, un, qs, wq, lane, wacc, p_begin, p_end); break;
    }
}

// ------------------------------------------------------------------------------------------------------------
// The fp32 path (ADMM_STORAGE_FP32_3XTF32): 3xTF32 with the big operand split ON CHIP INTO TENSOR MEMORY.
//
//   warp 0        TMA producer: raw fp32 tile of the big operand [128 rows][32] + the small operand [hi ; lo] stacked
//                 as ONE [2 n_mma][32] K-major tile
//   warps 2-5     converter: thread = one row.  Reads its 128 B from the swizzled smem tile, splits every value into
//                 hi = tf32_rna(x), lo = tf32_rna(x - hi) and writes both with tcgen05.st into a 2-deep TMEM ring
//                 (the A operand of the MMAs: lanes = rows, 32 columns = the k-block)
//   warp 1        UMMA issuer, per 8-element k-step TWO instructions (measured: a tf32 MMA of M=128 costs ~120 cycles
//                 for any N <= 192, so stacking [hi ; lo] along N is free):
//                     D[:, 0:2n)  += A_hi . [B_hi ; B_lo]^T      (main | small)
//                     D[:, n:2n)  += A_lo . B_hi^T               (small)
//   warps 6-13    drain + epilogue: tcgen05.mma adds with truncation (measured: every product is cut 2 bits below the
//                 accumulator's ulp and the sum is cut toward zero: a bias of ~0.45 ulp per MMA that is coherent over
//                 the iterations).  The MAIN accumulator is therefore read AND CLEARED every `chunk_kb` k-blocks and
//                 summed in fp32 registers with round-to-nearest FADDs; the MMAs always accumulate.  Two D regions
//                 alternate so the drain of chunk c overlaps the MMAs of chunk c+1.  The small (2^-11) terms stay in
//                 TMEM for the whole unit.
// TMEM columns: region 0 [0, 2n) | region 1 [2n, 4n) | A ring [384, 512) = 2 x (hi 32 | lo 32);   n = n_mma <= 96.
constexpr int kF32Warps = 23;              // TMA, MMA, 4 converter, 8 drain, 8 epilogue, second MMA issuer
constexpr int kMma2Warp = 22;
constexpr int kF32Threads = kF32Warps * 32;
constexpr int kF32MaxMmaN = 96;
constexpr int kAcol = 384;
constexpr int kConvWarp0 = 2, kDrainWarp0 = 6, kEpiWarp0 = 14;    // first warp of each role (4 consecutive warps cover the 4 TMEM lane quarters)
constexpr int kMaxAStages = 8, kMaxBStages = 4;

struct CtrlF32 {
    uint64_t sa_full[kMaxAStages];     // raw fp32 tile of the big operand landed in smem      (TMA -> converter)
    uint64_t sa_empty[kMaxAStages];    // converter has it in registers                         (converter -> TMA)
    uint64_t sb_full[kMaxBStages];     // small operand [hi ; lo] landed in smem                (TMA -> MMA)
    uint64_t sb_empty[kMaxBStages];    // MMAs that read it completed                           (MMA commit -> TMA)
    uint64_t a_full[2];                // hi | lo of a k-block are in TMEM                      (converter -> MMA)
    uint64_t a_empty[2];               //                                                       (MMA commit -> converter)
    uint64_t d_full[2];                // a chunk of MMAs into D region a completed             (MMA commit -> drain)
    uint64_t d_empty[2];               // region read and cleared                               (drain -> MMA)
    uint64_t q_full;                   // master sums of a unit staged in qs                    (drain -> epilogue)
    uint64_t q_empty;                  //                                                       (epilogue -> drain)
    uint32_t tmem_base;
    uint32_t pad;
};
__host__ __device__ inline int f32_b_bytes(int n_mma) { return 2 * n_mma * kBlockK * 4; }
__host__ __device__ inline int f32_q_bytes(int n_mma) { return n_mma * kTileM * 4; }        // staged accumulator tile
// per-warp partial sums [8 warps][n_mma][8]: only launches that sum something (residuals at a check, hinges of the objective)
// carve it out of shared memory; the others spend those 24 KB on one more stage of the big operand
__host__ __device__ inline bool f32_needs_acc(const TcLaunch& L) {
    return L.epi == EPI_OBJECTIVE || (L.epi == EPI_K3_STATE && L.ep.resid_partial != nullptr);
}
__host__ __device__ inline int f32_acc_bytes(int n_mma, bool need) { return need ? 8 * n_mma * 8 * 4 : 0; }
// B ring: 4 stages when the A ring still gets 3 (measured at config 1: A depth 3..5 makes no difference, B depth 2 / 3 / 4
// gives 120 / 107 / 104 us for K1: the L2-resident small operand arrives as 2 x n_mma rows of 128 B and has the longer latency)
__host__ __device__ inline int f32_b_stages(int n_mma, bool acc) {
    const int fixed = 1024 + (int)sizeof(CtrlF32) + f32_q_bytes(n_mma) + f32_acc_bytes(n_mma, acc);
    return (fixed + 4 * f32_b_bytes(n_mma) + 3 * kTileBytes <= kSmemLimit) ? 4 : 3;
}
__host__ __device__ inline int f32_a_stages(int n_mma, bool acc, int n_sb) {
    int s = (kSmemLimit - 1024 - (int)sizeof(CtrlF32) - f32_q_bytes(n_mma) - f32_acc_bytes(n_mma, acc) -
             n_sb * f32_b_bytes(n_mma)) / kTileBytes;
    return s > kMaxAStages ? kMaxAStages : s;
}

// iterator over the (unit, k-block) sequence of this CTA
struct KbIter {
    int u, kb, kb_count;
    __device__ __forceinline__ void start(const TcLaunch& L, int u0, int u_end) {
        u = u0; kb = 0; kb_count = (u0 < u_end) ? L.units[u0].kb_count : 0;
    }
    __device__ __forceinline__ void next(const TcLaunch& L, int u_end) {
        if (++kb == kb_count) { ++u; kb = 0; kb_count = (u < u_end) ? L.units[u].kb_count : 0; }
    }
};

__global__ void __launch_bounds__(kF32Threads, 1) admm_contract_f32_kernel(const __grid_constant__ TcLaunch L) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int n_mma = L.ep.n_mma;
    const int bbytes = f32_b_bytes(n_mma);
    const int n_sa = L.n_sa;
    const int n_sb = L.n_sb;
    uint8_t* a_ring = smem;                                   // n_sa x 16 KB (1024-aligned)
    uint8_t* b_ring = smem + n_sa * kTileBytes;               // n_sb x bbytes (multiple of 1024: n_mma % 16 == 0)
    float* qs = reinterpret_cast<float*>(b_ring + n_sb * bbytes);
    float* acc = qs + n_mma * kTileM;
    const bool need_acc = f32_needs_acc(L);
    CtrlF32* ctrl = reinterpret_cast<CtrlF32*>(reinterpret_cast<uint8_t*>(acc) + f32_acc_bytes(n_mma, need_acc));

    const int unit_begin = L.cta_unit_begin[blockIdx.x];
    const int unit_end = L.cta_unit_begin[blockIdx.x + 1];
    const int chunk_kb = L.chunk_kb;
    const int n_act = eff_nact(L.ep);
    if (n_act <= 0) return;                               // the whole pass froze since the host sized this launch

    if (threadIdx.x == 0) {
        // sa_empty: released by the 4 converter warps (3xTF32: the raw tile is in registers) or by the MMA commit (direct mode)
        for (int i = 0; i < n_sa; ++i) { tc::mbar_init(&ctrl->sa_full[i], 1); tc::mbar_init(&ctrl->sa_empty[i], L.mma_passes == 3 ? 4 : 1); }
        for (int i = 0; i < n_sb; ++i) { tc::mbar_init(&ctrl->sb_full[i], 1); tc::mbar_init(&ctrl->sb_empty[i], 1); }
        for (int i = 0; i < 2; ++i) {
            tc::mbar_init(&ctrl->a_full[i], 4);
            tc::mbar_init(&ctrl->a_empty[i], 1);
            tc::mbar_init(&ctrl->d_full[i], (L.mma_passes == 3 && L.chunk_kb == 1) ? 2 : 1);      // one arrival per MMA issuer
            tc::mbar_init(&ctrl->d_empty[i], 8);
        }
        tc::mbar_init(&ctrl->q_full, 8);
        tc::mbar_init(&ctrl->q_empty, 8);
        tc::fence_barrier_init();
        tc::tma_prefetch_desc(&L.map_big);
        tc::tma_prefetch_desc(&L.map_small_hi);
        tc::tma_prefetch_desc(&L.map_small_lo);
    }
    for (int i = threadIdx.x; i < f32_acc_bytes(n_mma, need_acc) / 4; i += kF32Threads) acc[i] = 0.0f;
    if (warp == 1) tc::tmem_alloc(&ctrl->tmem_base, 512);
    tc::tcgen05_fence_before();
    __syncthreads();
    tc::tcgen05_fence_after();
    const uint32_t tmem_base = ctrl->tmem_base;
    if (warp >= kDrainWarp0 && warp < kEpiWarp0) {
        // the MMAs always accumulate: clear both D regions once (this warp's lane quarter, its half of 384 columns)
        const uint32_t lane_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
        uint32_t z[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) z[i] = 0u;
        const int c_lo = ((warp - kDrainWarp0) >> 2) * (kAcol / 2);
        for (int c = c_lo; c < c_lo + kAcol / 2; c += 16) tc::tmem_st16(lane_addr + c, z);
        tc::tmem_st_wait();
    }
    tc::tcgen05_fence_before();
    __syncthreads();
    tc::tcgen05_fence_after();

    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer: two independent rings, one polling lane
        if (lane == 0) {
            // the unit record is read from global memory ONCE per unit and kept in registers (reading L.units[] for every
            // k-block put a dependent global load in front of every TMA issue)
            int ua = unit_begin, ub = unit_begin, kba = 0, kbb = 0;
            TcUnit una = TcUnit{0, 0, 0, 0, 0, 0}, unb = una;
            if (unit_begin < unit_end) { una = L.units[unit_begin]; unb = una; }
            int arow = ((una.row0 >> 7) * L.big_kb_total + una.kb0) * kTileM;      // tile-major row of the next A tile
            int bk0 = unb.kb0 * L.kblk;                                             // element coordinate of the next B tile
            int sa = 0, sb = 0; uint32_t pha = 0, phb = 0;
            while (ua < unit_end || ub < unit_end) {
                if (ua < unit_end && tc::mbar_test_wait(&ctrl->sa_empty[sa], pha ^ 1)) {
                    // one 16 KB tile of the tile-major big operand (rows past the end of the matrix are stored as zeros)
                    tc::mbar_arrive_expect_tx(&ctrl->sa_full[sa], kTileBytes);
                    tc::tma_load_2d(a_ring + sa * kTileBytes, &L.map_big128, &ctrl->sa_full[sa], 0, arow, tc::kEvictFirst);
                    arow += kTileM;
                    if (++kba == una.kb_count) {
                        kba = 0;
                        if (++ua < unit_end) { una = L.units[ua]; arow = ((una.row0 >> 7) * L.big_kb_total + una.kb0) * kTileM; }
                    }
                    if (++sa == n_sa) { sa = 0; pha ^= 1; }
                }
                if (ub < unit_end && tc::mbar_test_wait(&ctrl->sb_empty[sb], phb ^ 1)) {
                    tc::mbar_arrive_expect_tx(&ctrl->sb_full[sb], bbytes);
                    tc::tma_load_2d(b_ring + sb * bbytes, &L.map_small_hi, &ctrl->sb_full[sb], bk0, 0, tc::kEvictLast);
                    tc::tma_load_2d(b_ring + sb * bbytes + bbytes / 2, &L.map_small_lo, &ctrl->sb_full[sb], bk0, 0, tc::kEvictLast);
                    bk0 += L.kblk;
                    if (++kbb == unb.kb_count) {
                        kbb = 0;
                        if (++ub < unit_end) { unb = L.units[ub]; bk0 = unb.kb0 * L.kblk; }
                    }
                    if (++sb == n_sb) { sb = 0; phb ^= 1; }
                }
            }
        }
    } else if (warp == 1 || warp == kMma2Warp) {
        // ------------------------------------------------------------ UMMA issuers (warp-uniform loop, one elected lane issues)
        // TWO issuing warps take the k-blocks in turn (even / odd): measured with clock64, one warp needs ~1200 cycles of
        // serial latency per k-block (three mbarrier probes ~130 each, fence + 8 MMAs + 3 commits ~530, bookkeeping) for 576
        // cycles of tensor work, so a single issuer kept the pipe half idle.  k-block parity = A-ring slot = parity of the (even-
        // depth) smem stages, so each of those barriers is always probed by the same warp and no phase goes unobserved; the D
        // regions are shared: both warps wait d_empty and both arrive on d_full (count 2), by commit after their last k-block
        // of the chunk or by a plain arrive when the chunk held none of theirs.
        const int mma_id = (warp == 1) ? 0 : 1;
        // direct modes keep ONE issuer: there the MMA warp also waits on the smem A ring, whose depth (3 at n_mma = 96) would have
        // to be cut to 2 to stay even, which costs more than the second issuer gains (measured: tf32 102 -> 123 us)
        // ... and a chunk of several k-blocks stays with ONE issuer too: two threads accumulating into the same D region do so in
        // an order the hardware does not fix, and the fp32 sums came out different from run to run (measured at drain_kb = 2)
        const bool two = L.mma_passes == 3 && chunk_kb == 1;
        int gkb = 0;                        // k-blocks seen so far (all units): its parity picks the issuer
        if (two || mma_id == 0) {
        const bool direct = L.mma_passes != 3;     // Phi already exact in the operand format (tf32 / bf16 storage): A straight from smem
        const uint32_t fmt = L.mma_kind == 1 ? 1u : 2u;
        const uint32_t idesc_wide = tc::umma_idesc(fmt, kTileM, (uint32_t)(2 * n_mma));
        const uint32_t idesc_one = tc::umma_idesc(fmt, kTileM, (uint32_t)n_mma);
        const uint64_t a_desc0 = tc::umma_desc_k_sw128(tc::smem_u32(a_ring));
        int sa = 0; uint32_t pha = 0;              // smem A ring (direct mode)
        const uint64_t b_desc0 = tc::umma_desc_k_sw128(tc::smem_u32(b_ring));
        const uint64_t b_step = (uint64_t)(bbytes >> 4);
        uint64_t b_desc = b_desc0;
        int sb = 0; uint32_t phb = 0;      // smem B ring
        int t = 0; uint32_t tph = 0;       // TMEM A ring
        int a = 0; uint32_t aph = 0;       // D region
        for (int u = unit_begin; u < unit_end; ++u) {
            const int kb_count = L.units[u].kb_count;
            const int ck = chunk_kb > 0 ? chunk_kb : kb_count;
            for (int kb0 = 0; kb0 < kb_count; kb0 += ck) {
                const int nkb = min(ck, kb_count - kb0);
                tc::mbar_wait(&ctrl->d_empty[a], aph ^ 1);
                const uint32_t d_main = tmem_base + a * 2 * n_mma;
                const uint32_t d_small = d_main + n_mma;
                // my last k-block of this chunk (-1: none): that is where my arrival on d_full goes
                int my_last = -1;
                for (int kb = nkb - 1; kb >= 0; --kb) if (!two || ((gkb + kb) & 1) == mma_id) { my_last = kb; break; }
                if (my_last < 0) { if (tc::elect_one()) tc::mbar_arrive(&ctrl->d_full[a]); __syncwarp(); }
                for (int kb = 0; kb < nkb; ++kb, ++gkb) {
                    const bool mine = !two || (gkb & 1) == mma_id;
                    if (!mine) {            // the other issuer's k-block: only keep the ring counters in step
                        b_desc += b_step;
                        if (++sb == n_sb) { sb = 0; phb ^= 1; b_desc = b_desc0; }
                        if (++sa == n_sa) { sa = 0; pha ^= 1; }
                        if (++t == 2) { t = 0; tph ^= 1; }
                        continue;
                    }
                    tc::mbar_wait(&ctrl->sb_full[sb], phb);     // the small operand landed (async proxy)
                    if (direct) {
                        tc::mbar_wait(&ctrl->sa_full[sa], pha); // the big operand's tile landed (async proxy): it IS the A operand
                        tc::tcgen05_fence_after();
                        const uint64_t a_desc = a_desc0 + (uint64_t)(sa * (kTileBytes >> 4));
                        if (tc::elect_one()) {
                            // one MMA per 32-byte k-step (8 tf32 / 16 bf16 elements): D[:, 0:2n) += A . [B_hi ; B_lo]^T
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                if (fmt == 1u) tc::umma_f16(d_main, a_desc + 2 * k, b_desc + 2 * k, idesc_wide, 1u);
                                else tc::umma_tf32(d_main, a_desc + 2 * k, b_desc + 2 * k, idesc_wide, 1u);
                            }
                            tc::umma_commit(&ctrl->sb_empty[sb]);
                            tc::umma_commit(&ctrl->sa_empty[sa]);
                            if (kb == my_last) tc::umma_commit(&ctrl->d_full[a]);
                        }
                        __syncwarp();
                    } else {
                    tc::mbar_wait(&ctrl->a_full[t], tph);       // the converter's hi/lo are in TMEM
                    tc::tcgen05_fence_after();
                    const uint32_t a_hi = tmem_base + kAcol + t * 64;
                    if (tc::elect_one()) {
#pragma unroll
                        for (int k = 0; k < kBlockK / 8; ++k) {
                            tc::umma_tf32_ts(d_main, a_hi + k * 8, b_desc + 2 * k, idesc_wide, 1u);
                            tc::umma_tf32_ts(d_small, a_hi + 32 + k * 8, b_desc + 2 * k, idesc_one, 1u);
                        }
                        tc::umma_commit(&ctrl->sb_empty[sb]);
                        tc::umma_commit(&ctrl->a_empty[t]);
                        if (kb == my_last) tc::umma_commit(&ctrl->d_full[a]);
                    }
                    __syncwarp();
                    }
                    b_desc += b_step;
                    if (++sb == n_sb) { sb = 0; phb ^= 1; b_desc = b_desc0; }
                    if (++sa == n_sa) { sa = 0; pha ^= 1; }
                    if (++t == 2) { t = 0; tph ^= 1; }
                }
                if (++a == 2) { a = 0; aph ^= 1; }
            }
        }
        }
    } else if (warp >= kConvWarp0 && warp < kDrainWarp0) {
        if (L.mma_passes == 3) {
        // ------------------------------------------------------------ converter: smem fp32 row -> TMEM hi | lo
        // hi = tf32_rna(x) (round to nearest: lo = x - hi is then symmetric in sign, so the tensor core's truncation of
        // lo's low bits is unbiased; with a truncated hi, lo >= 0 for Phi >= 0 and the products came out 2^-22 too small)
        const int q = warp & 3;                         // TMEM lane quarter of this warp
        const int lrow = q * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16) + kAcol;
        int sa = 0; uint32_t pha = 0;
        int t = 0; uint32_t tph = 0;
        for (int u = unit_begin; u < unit_end; ++u) {
            const int kbc = L.units[u].kb_count;
            for (int kb = 0; kb < kbc; ++kb) {
                tc::mbar_wait(&ctrl->sa_full[sa], pha);
                const uint8_t* row = a_ring + sa * kTileBytes + lrow * 128;
                float4 v[8];
#pragma unroll
                for (int c = 0; c < 8; ++c) v[c] = *reinterpret_cast<const float4*>(row + ((c ^ (lrow & 7)) << 4));
                __syncwarp();
                if (lane == 0) tc::mbar_arrive(&ctrl->sa_empty[sa]);      // the raw tile is in registers: free the slot
                tc::mbar_wait(&ctrl->a_empty[t], tph ^ 1);
                tc::tcgen05_fence_after();
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    uint32_t hi[16], lo[16];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const float4 x = v[h * 4 + c];
                        const float xs[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const float hf = tc::tf32_rna(xs[e]);
                            hi[c * 4 + e] = __float_as_uint(hf);
                            lo[c * 4 + e] = __float_as_uint(xs[e] - hf);
                        }
                    }
                    tc::tmem_st16(lane_addr + t * 64 + h * 16, hi);
                    tc::tmem_st16(lane_addr + t * 64 + 32 + h * 16, lo);
                }
                tc::tmem_st_wait();
                tc::tcgen05_fence_before();
                __syncwarp();
                if (lane == 0) tc::mbar_arrive(&ctrl->a_full[t]);
                if (++sa == n_sa) { sa = 0; pha ^= 1; }
                if (++t == 2) { t = 0; tph ^= 1; }
            }
        }
        }
    } else if (warp >= kDrainWarp0 && warp < kEpiWarp0) {
        // ------------------------------------------------------------ drain (row = TMEM lane): TMEM -> fp32 master sums -> qs
        const int ew = warp & 3;
        const int n16 = n_mma / 16;
        const int half = (warp - kDrainWarp0) >> 2;
        const int cbeg = half == 0 ? 0 : (n16 + 1) / 2;          // first 16-column group of this warp
        const int cend = half == 0 ? (n16 + 1) / 2 : n16;        // at most 3 groups (n_mma <= 96)
        const int lrow = ew * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(ew * 32) << 16);
        uint32_t zero[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) zero[i] = 0u;
        int a = 0; uint32_t aph = 0;
        uint32_t qph = 0;
        for (int u = unit_begin; u < unit_end; ++u) {
            const int kb_count = L.units[u].kb_count;
            float master[48];
#pragma unroll
            for (int i = 0; i < 48; ++i) master[i] = 0.0f;
            const int ck = chunk_kb > 0 ? chunk_kb : kb_count;
            const int nchunks = (kb_count + ck - 1) / ck;
            for (int ci = 0; ci < nchunks; ++ci) {
                tc::mbar_wait(&ctrl->d_full[a], aph);
                tc::tcgen05_fence_after();
                const uint32_t d_main = lane_addr + a * 2 * n_mma;
                const bool with_small = ci + 2 >= nchunks;       // last use of this region in the unit
#pragma unroll
                for (int cc = 0; cc < 3; ++cc) {
                    if (cbeg + cc < cend) {
                        uint32_t r[16];
                        tc::tmem_ld16(d_main + (cbeg + cc) * 16, r);
                        tc::tmem_ld_wait(r);
#pragma unroll
                        for (int jj = 0; jj < 16; ++jj) master[cc * 16 + jj] += __uint_as_float(r[jj]);
                        tc::tmem_st16(d_main + (cbeg + cc) * 16, zero);
                        if (with_small) {
                            tc::tmem_ld16(d_main + n_mma + (cbeg + cc) * 16, r);
                            tc::tmem_ld_wait(r);
#pragma unroll
                            for (int jj = 0; jj < 16; ++jj) master[cc * 16 + jj] += __uint_as_float(r[jj]);
                            tc::tmem_st16(d_main + n_mma + (cbeg + cc) * 16, zero);
                        }
                    }
                }
                tc::tmem_st_wait();
                tc::tcgen05_fence_before();
                __syncwarp();
                if (lane == 0) tc::mbar_arrive(&ctrl->d_empty[a]);
                if (++a == 2) { a = 0; aph ^= 1; }
            }
            // hand the finished tile to the epilogue warps and go on draining the next unit.  De-bias: every
            // drained chunk came out of the tensor core low by ~debias of its value (the accumulator adds with truncation), so the
            // sum of the chunks is low by the same fraction: one FMA per output puts it back.
            tc::mbar_wait(&ctrl->q_empty, qph ^ 1);
            const float kappa = L.debias;
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
                if (cbeg + cc < cend) {
#pragma unroll
                    for (int jj = 0; jj < 16; ++jj)
                        qs[((cbeg + cc) * 16 + jj) * kTileM + lrow] = fmaf(master[cc * 16 + jj], kappa, master[cc * 16 + jj]);
                }
            }
            __syncwarp();
            if (lane == 0) tc::mbar_arrive(&ctrl->q_full);
            qph ^= 1;
        }
    } else if (warp >= kEpiWarp0) {
        // ------------------------------------------------------------ epilogue warps: qs -> global, concurrent with the next unit
        const int wq = (warp - kEpiWarp0) & 3;           // row quarter
        const int ph_half = (warp - kEpiWarp0) >> 2;     // which half of the plans
        const int p_mid = (n_act + 1) / 2;
        const int p_begin = ph_half == 0 ? 0 : p_mid;
        const int p_end = ph_half == 0 ? p_mid : n_act;
        uint32_t qph = 0;
        if (unit_begin < unit_end) prefetch_s1_tile(L, L.units[unit_begin], wq, lane, p_begin, p_end);
        for (int u = unit_begin; u < unit_end; ++u) {
            const TcUnit un = L.units[u];
            if (u + 1 < unit_end) prefetch_s1_tile(L, L.units[u + 1], wq, lane, p_begin, p_end);
            tc::mbar_wait(&ctrl->q_full, qph);
            epilogue_unit(L, un, qs, wq, lane, acc + (warp - kEpiWarp0) * n_mma * 8, p_begin, p_end);
            __syncwarp();
            if (lane == 0) tc::mbar_arrive(&ctrl->q_empty);
            qph ^= 1;
        }
    }

    __syncthreads();
    if (L.epi == EPI_K3_STATE && L.ep.resid_partial != nullptr) {
        for (int i = threadIdx.x; i < n_act * kNumResid; i += kF32Threads) {
            const int p = i / kNumResid, t = i % kNumResid;
            float v = 0.f;
            for (int w = 0; w < 8; ++w) v += acc[(w * n_mma + p) * 8 + t];
            L.ep.resid_partial[((int64_t)blockIdx.x * kMaxBpad + L.ep.slot0 + p) * kNumResid + t] = v;
        }
    } else if (L.epi == EPI_OBJECTIVE) {
        for (int i = threadIdx.x; i < n_act * kMaxClasses; i += kF32Threads) {
            const int p = i / kMaxClasses, k = i % kMaxClasses;
            double v = 0.0;
            for (int w = 0; w < 8; ++w) v += (double)acc[(w * n_mma + p) * 8 + k];
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
    cudaError_t e = cudaFuncSetAttribute(admm_contract_f32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(admm_contract_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
    if (e != cudaSuccess) {
        h->err = std::string("cudaFuncSetAttribute(max dynamic smem): ") + cudaGetErrorString(e);
        return ADMM_ECUDA;
    }
    return ADMM_OK;
}

// 2-D fp32 tensor [rows][cols] with row stride ld_elems, box = {32 cols (128 B), box_rows}, 128-byte swizzle,
// out-of-bounds elements read as zero.
admm_status tc_make_map(admm_handle* h, CUtensorMap* out, const void* base, int64_t rows, int64_t cols,
                        int64_t ld_elems, int box_rows, int elem_bytes) {
    cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t gstride[1] = {(cuuint64_t)ld_elems * elem_bytes};
    cuuint32_t box[2] = {(cuuint32_t)(128 / elem_bytes), (cuuint32_t)box_rows};       // 128-byte rows
    cuuint32_t estr[2] = {1, 1};
    CUresult r = g_encode(out, elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                          const_cast<void*>(base), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
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
    if ((kSmemLimit - 1024 - (int)sizeof(Ctrl) - acc_bytes(n_mma)) / stage_bytes(n_mma) < 2) {
        h->err = "tc_launch: fewer than 2 pipeline stages fit in shared memory";
        return ADMM_EINVAL;
    }
    if (L.mma_passes == 3 || n_mma <= kF32MaxMmaN) {
        // the staged kernel: 3xTF32 (converter + TS MMAs), or "direct" for tf32 / bf16 storage (A from shared memory)
        if (n_mma > kF32MaxMmaN) { h->err = "tc_launch: the fp32 path needs n_mma <= 96"; return ADMM_EINVAL; }
        TcLaunch L2 = L;
        const bool acc = f32_needs_acc(L);
        L2.n_sb = f32_b_stages(n_mma, acc);
        // the two MMA issuers take the chunks in turn and only probe the barriers of their own k-blocks: every ring they wait on
        // must have an EVEN depth, so that a stage is always consumed by the same warp and no mbarrier phase goes unobserved
        // (a parity probe cannot tell "two phases behind" from "done").  3xTF32 mode only (direct modes have one issuer): B ring 4 or 2;
        // the A rings it waits on are the 2 TMEM slots.
        if (L.mma_passes == 3 && L2.n_sb == 3) L2.n_sb = 2;
        L2.n_sa = f32_a_stages(n_mma, acc, L2.n_sb);
        if (L2.n_sa < 2) { h->err = "tc_launch: fewer than 2 pipeline stages fit in shared memory"; return ADMM_EINVAL; }
        admm_contract_f32_kernel<<<L.grid, kF32Threads, kSmemLimit, h->stream>>>(L2);
    } else {
        admm_contract_kernel<<<L.grid, 320, kSmemLimit, h->stream>>>(L);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        h->err = std::string("admm_contract_kernel launch: ") + cudaGetErrorString(e);
        return ADMM_ECUDA;
    }
    h->launch_count++;
    return ADMM_OK;
}
