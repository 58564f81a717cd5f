// Everything on the hot path that is not a tcgen05 contraction: the S^-1 apply with fused epilogue-2
// (K2a/K2b), the stopping rule, state start-up / read-out, setup helpers, and the plain-FFMA
// cross-check versions of K1/K3 (ADMM_PATH_SIMT).
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include "admm_internal.h"
#include "epilogue.cuh"

namespace {

inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ------------------------------------------------------------------------------------------ setup helpers
__global__ void transpose_kernel(const float* __restrict__ src, int64_t rows, int64_t cols, int64_t ld_src,
                                 float* __restrict__ dst, int64_t ld_dst) {
    __shared__ float tile[32][33];
    const int64_t c0 = (int64_t)blockIdx.x * 32, r0 = (int64_t)blockIdx.y * 32;
    for (int y = threadIdx.y; y < 32; y += 8) {
        int64_t r = r0 + y, c = c0 + threadIdx.x;
        tile[y][threadIdx.x] = (r < rows && c < cols) ? src[r * ld_src + c] : 0.0f;
    }
    __syncthreads();
    for (int y = threadIdx.y; y < 32; y += 8) {
        int64_t c = c0 + y, r = r0 + threadIdx.x;
        if (c < cols && r < rows) dst[c * ld_dst + r] = tile[threadIdx.x][y];
    }
}

// Tile-major copy of a big operand for the tcgen05 contractions: dst[(rt * KB + kb)][128][32] = the 128 x 32 block of
// rows rt*128.., columns kb*32.. of X (zero outside), X = src (TRANSPOSE = false) or src^T (true).  One TMA box of a
// contraction kernel is then ONE contiguous 16 KB burst and a CTA walking k reads sequential memory: with the row-major
// layout each box was 128 pieces of 128 B a row stride apart (1.8 MB for Phi^T at config 2: one DRAM page and one TLB
// entry per piece).  Block = one tile, 256 threads.
template <bool TRANSPOSE>
__global__ void __launch_bounds__(256) pack_tiles_kernel(const float* __restrict__ src, int64_t src_rows, int64_t src_cols,
                                                         int64_t ld_src, float* __restrict__ dst, int64_t KB) {
    const int64_t kb = blockIdx.x, rt = blockIdx.y;
    float* out = dst + ((rt * KB + kb) * kTileM) * kBlockK;
    if (!TRANSPOSE) {
        // X = src: rows rt*128 + r, cols kb*32 + c
        for (int i = threadIdx.x; i < kTileM * kBlockK; i += 256) {
            const int r = i >> 5, c = i & 31;
            const int64_t row = rt * kTileM + r, col = kb * kBlockK + c;
            out[i] = (row < src_rows && col < src_cols) ? src[row * ld_src + col] : 0.0f;
        }
    } else {
        // X = src^T: X[j][i] = src[i][j]; tile rows j = rt*128 + r (src columns), tile cols i = kb*32 + c (src rows)
        __shared__ float t[kBlockK][kTileM + 1];
        for (int i = threadIdx.x; i < kTileM * kBlockK; i += 256) {
            const int c = i >> 7, r = i & 127;                       // c: src row within the block, r: src column
            const int64_t srow = kb * kBlockK + c, scol = rt * kTileM + r;
            t[c][r] = (srow < src_rows && scol < src_cols) ? src[srow * ld_src + scol] : 0.0f;
        }
        __syncthreads();
        for (int i = threadIdx.x; i < kTileM * kBlockK; i += 256) {
            const int r = i >> 5, c = i & 31;
            out[i] = t[c][r];
        }
    }
}

// out[r][j] = a_cls[class(row0 + r)] * phi[row0 + r][j]  in fp64 (operand of the fp64 SYRK)
__global__ void scale_rows_kernel(const float* __restrict__ phi, int64_t ld, int64_t row0, int64_t rows, int64_t n,
                                  const uint8_t* __restrict__ cls, const double* __restrict__ a_cls, double* __restrict__ out) {
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= rows * n) return;
    int64_t r = idx / n, j = idx % n;
    out[idx] = a_cls[cls[row0 + r]] * (double)phi[(row0 + r) * ld + j];
}

__global__ void round_tf32_kernel(float* x, int64_t count) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) x[i] = tc::tf32_rn(x[i]);
}

__global__ void round_bf16_kernel(float* x, int64_t count) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) x[i] = __bfloat162float(__float2bfloat16_rn(x[i]));
}

// bf16 tile-major copy: dst[(rt * KB + kb)][128][64] bf16 (128-byte rows of 64 elements); src holds values already on
// the bf16 grid (round_bf16_kernel), so the conversion is exact.
template <bool TRANSPOSE>
__global__ void __launch_bounds__(256) pack_tiles_bf16_kernel(const float* __restrict__ src, int64_t src_rows, int64_t src_cols,
                                                              int64_t ld_src, __nv_bfloat16* __restrict__ dst, int64_t KB) {
    constexpr int KE = 64;
    const int64_t kb = blockIdx.x, rt = blockIdx.y;
    __nv_bfloat16* out = dst + ((rt * KB + kb) * kTileM) * KE;
    if (!TRANSPOSE) {
        for (int i = threadIdx.x; i < kTileM * KE; i += 256) {
            const int r = i >> 6, c = i & 63;
            const int64_t row = rt * kTileM + r, col = kb * KE + c;
            out[i] = __float2bfloat16_rn((row < src_rows && col < src_cols) ? src[row * ld_src + col] : 0.0f);
        }
    } else {
        __shared__ float t[KE][kTileM + 1];
        for (int i = threadIdx.x; i < kTileM * KE; i += 256) {
            const int c = i >> 7, r = i & 127;
            const int64_t srow = kb * KE + c, scol = rt * kTileM + r;
            t[c][r] = (srow < src_rows && scol < src_cols) ? src[srow * ld_src + scol] : 0.0f;
        }
        __syncthreads();
        for (int i = threadIdx.x; i < kTileM * KE; i += 256) {
            const int r = i >> 6, c = i & 63;
            out[i] = __float2bfloat16_rn(t[c][r]);
        }
    }
}

// R_j = 1/sqrt(M_jj) (1 if the row of A D is zero)
__global__ void make_R_kernel(const double* __restrict__ M, int64_t n, double* __restrict__ R) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) { double d = M[j * n + j]; R[j] = d > 0.0 ? 1.0 / sqrt(d) : 1.0; }
}
// S = I + R M R, lower triangle (column-major lower == row-major upper; M is symmetric after the fill below)
__global__ void finish_S_kernel(double* __restrict__ M, int64_t n, const double* __restrict__ R) {
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * n) return;
    int64_t r = idx / n, c = idx % n;
    M[idx] = R[r] * M[idx] * R[c] + (r == c ? 1.0 : 0.0);
}
// copy the computed triangle onto the other one: A[r][c] (c > r) <- A[c][r]
__global__ void symmetrize_kernel(double* __restrict__ A, int64_t n, int from_lower_rowmajor) {
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * n) return;
    int64_t r = idx / n, c = idx % n;
    if (from_lower_rowmajor) { if (c > r) A[r * n + c] = A[c * n + r]; }
    else { if (c < r) A[r * n + c] = A[c * n + r]; }
}

// counts[p][k] = number of ACTIVE rows of class k in plan p
__global__ void count_active_kernel(const uint32_t* __restrict__ mask, int64_t mask_words, const uint8_t* __restrict__ cls,
                                    int64_t N, int32_t* __restrict__ counts) {
    const int p = blockIdx.x;
    int local[kMaxClasses];
    for (int k = 0; k < kMaxClasses; ++k) local[k] = 0;
    for (int64_t i = threadIdx.x; i < N; i += blockDim.x) {
        uint32_t w = mask ? mask[(int64_t)p * mask_words + (i >> 5)] : 0xFFFFFFFFu;
        if ((w >> (i & 31)) & 1u) local[cls[i]]++;
    }
    __shared__ int sh[kMaxClasses];
    if (threadIdx.x < kMaxClasses) sh[threadIdx.x] = 0;
    __syncthreads();
    for (int k = 0; k < kMaxClasses; ++k) {
        int v = local[k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0 && v) atomicAdd(&sh[k], v);
    }
    __syncthreads();
    if (threadIdx.x < kMaxClasses) counts[p * kMaxClasses + threadIdx.x] = sh[threadIdx.x];
}

// ------------------------------------------------------------------------------------------ state start-up / read-out
__device__ __forceinline__ float mask_ub(const EpiParams& ep, int cls, int slot, int64_t row) {
    bool on = true;
    if (ep.mask) on = (ep.mask[(int64_t)ep.slot_plan[slot] * ep.mask_words + (row >> 5)] >> (row & 31)) & 1u;
    return on ? ep.utab[cls * kMaxBpad + slot] : 0.0f;
}

// G = a (2 z1 - s1 - c/rho) from the current s1 (all-zero start: G = -a c/rho)
__global__ void emit_g_kernel(const EpiParams ep, int Bact) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = ep.slot0 + blockIdx.y;
    if (i >= ep.N || (int)blockIdx.y >= Bact) return;
    int cls = ep.point_class[i];
    float ub = mask_ub(ep, cls, p, i);
    float cr = ep.crtab[cls * kMaxBpad + p];
    float s = ep.s1[(int64_t)p * ep.ldN + i];
    float z = fminf(fmaxf(s, 0.f), ub);
    float g = ep.a_cls[cls] * (2.f * z - s - cr);
    emit_small(ep.g_hi, ep.g_lo, (int64_t)p * ep.ldN, i, g, ep.small_bf16 != 0);
}

__global__ void state_out_kernel(const EpiParams ep, int slot, const double* __restrict__ s2, const double* __restrict__ R,
                                 const double* __restrict__ beta_tab, float* z1, float* y1, double* z2, double* y2) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const double beta = beta_tab[slot];
    if (i < ep.N && (z1 || y1)) {
        int cls = ep.point_class[i];
        float ub = mask_ub(ep, cls, slot, i);
        float s = ep.s1[(int64_t)slot * ep.ldN + i];
        float z = fminf(fmaxf(s, 0.f), ub);
        if (z1) z1[i] = z;
        if (y1) y1[i] = s - z;
    }
    if (i < ep.n && (z2 || y2)) {
        double s = s2[(int64_t)slot * ep.ldn + i];
        double z = fmin(s, R[i] * beta);
        if (z2) z2[i] = z;
        if (y2) y2[i] = s - z;
    }
}

// t = rho R max(s2 - R beta, 0): fp32 output + tf32 hi/lo operand of the objective contraction
__global__ void make_t_kernel(const double* __restrict__ s2, const double* __restrict__ R, const double* __restrict__ Rb,
                              const double* __restrict__ beta, const double* __restrict__ rho, int64_t n, int64_t ldn, int Bact,
                              void* __restrict__ t_hi, void* __restrict__ t_lo, float* __restrict__ t_f32, int bf16) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;
    if (j >= n || p >= Bact) return;
    double y2 = fmax(s2[(int64_t)p * ldn + j] - Rb[j] * beta[p], 0.0);          // b_hat_j = R_j w_BOT on the rows that carry it (Eq. 13)
    double t = rho[p] * R[j] * y2;
    emit_small(t_hi, t_lo, (int64_t)p * ldn, j, t, bf16 != 0);
    t_f32[(int64_t)p * ldn + j] = (float)t;
}

// ------------------------------------------------------------------------------------------ K2a: rhs of Eq. (6)
// rhs[p][j] = R_j * sum_slots partial[slot][p][j - 128 mt]  -  (2 z2 - s2)[p][j]     (fp64)
__global__ void k2a_kernel(const float* __restrict__ partial, const int32_t* __restrict__ mtile_slot_begin, int n_mma,
                           const double* __restrict__ s2, const double* __restrict__ R, const double* __restrict__ Rb,
                           const double* __restrict__ beta, int64_t n, int64_t ldn, int slot0, int nact,
                           const int32_t* __restrict__ bact_dev, double* __restrict__ rhs) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;                       // index inside this contraction pass
    if (bact_dev) nact = min(nact, *bact_dev - slot0);
    if (j >= n || p >= nact) return;
    int mt = (int)(j / kTileM), jl = (int)(j % kTileM);
    double w = 0.0;
    for (int s = mtile_slot_begin[mt]; s < mtile_slot_begin[mt + 1]; ++s)
        w += (double)partial[((int64_t)s * n_mma + p) * kTileM + jl];
    const int gs = slot0 + p;
    double sv = s2[(int64_t)gs * ldn + j];
    double z = fmin(sv, Rb[j] * beta[gs]);
    rhs[(int64_t)gs * ldn + j] = R[j] * w - (2.0 * z - sv);
}

// ------------------------------------------------------------------------------------------ K2b: v = S^-1 rhs + epilogue-2
// Eq. (6): v = S^-1 (A r1 - r2) with the explicit fp64 inverse computed once at setup (:91, :165).
// fp64 on purpose (SURVEY H-a): this product is ~1 % of the flops of an iteration and its
// rounding error, amplified by cond(S), is what dominates the iterate error when it is done in fp32.
// tcgen05 has no fp64 kind; the fp64 tensor path of sm_100 is mma.sync m8n8k4 (DMMA), used here directly.
//
// Block = WJ x 2 warps; warp tile = 16 rows (time variables j) x 48 plans = 2 x 6 DMMA fragments; block tile = 16 WJ x 96.
// K is walked in chunks of 64 through a cp.async ring (as deep as ~200 KB allows); both operands are K-contiguous in memory
// (Sinv[j][k] row-major with padded row stride, rhs[p][k] plan-major), rows padded to 68 doubles => conflict-free LDS.64.
// Epilogue (4b)/(4c) on block 2 in single-state form: s2+ = z2 + v, z2 = min(s2, R beta); emits V = R o v (tf32 hi/lo).
constexpr int K2_TP = 96, K2_KC = 64, K2_LD = K2_KC + 4;       // 64-column chunks: half as many barrier rounds as 32
constexpr int K2_TPR = K2_KC / 2, K2_RPP = 256 / K2_TPR;        // loader: threads per row (16-byte pieces), rows per pass
// ring depth: as many 32-column chunks as fit in ~200 KB (the operands come from L2 / HBM at ~1 us latency and the
// DMMA work per chunk is a few hundred cycles: bytes in flight are what sets the speed)
#ifndef K2_SMEM_KB
#define K2_SMEM_KB 200        // (226 gives 32- and 40-row tiles a third stage: measured 4 % slower at 32 rows, 0-3 % faster at 40)
#endif
__host__ __device__ constexpr int k2_stages(int TJ) { return (K2_SMEM_KB * 1024) / ((TJ + K2_TP) * K2_LD * 8) > 8 ? 8 : (K2_SMEM_KB * 1024) / ((TJ + K2_TP) * K2_LD * 8); }

__device__ __forceinline__ void cp_async16_zfill(void* smem_dst, const void* gsrc, bool ok) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    const int sz = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;" ::"r"(d), "l"(gsrc), "r"(sz), "l"(tc::kEvictLast) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

template <int WJ, int RA>
__global__ void __launch_bounds__(256) k2b_kernel(const double* __restrict__ Sinv, int64_t lds,
                                                  const double* __restrict__ rhs, double* __restrict__ s2,
                                                  const double* __restrict__ R, const double* __restrict__ Rb,
                                                  const double* __restrict__ beta,
                                                  int64_t n, int64_t ldn, int Bact, const int32_t* __restrict__ bact_dev,
                                                  void* __restrict__ v_hi, void* __restrict__ v_lo, int bf16,
                                                  double* __restrict__ resid_partial) {
    if (bact_dev) Bact = min(Bact, *bact_dev);             // the host's bound lags the device by up to one check interval
    if ((int)blockIdx.y * K2_TP >= Bact) return;
    // 8 warps = WJ row groups x 2 plan halves x KS k-slices (a lone warp per scheduler cannot hide the DMMA issue
    // latency: measured 14 % pipe utilisation with 2 warps per block); the k-slices are summed through shared memory.
    // RA = 8-row DMMA fragments per warp tile along j: warp tile = 8 RA rows x 48 plans = RA x 6 fragments.  RA = 4 (32 x 48) issues
    // 10 LDS.64 per 24 DMMAs where RA = 2 issues 8 per 12: at a 64-row block tile the kernel was shared-memory-bandwidth bound.
    constexpr int RW = 8 * RA, TJ = RW * WJ, NT = 256, ROWS = TJ + K2_TP, KS = 4 / WJ, K2_STAGES = k2_stages(TJ);
    extern __shared__ __align__(16) double k2sm[];        // [K2_STAGES][ROWS][K2_LD]; reused after the main loop
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wj = warp % WJ, wp = (warp / WJ) & 1, kq = warp / (2 * WJ);
    const int g = lane >> 2, q = lane & 3;
    const int64_t j0 = (int64_t)blockIdx.x * TJ;
    const int p0 = blockIdx.y * K2_TP;
    const int nchunks = (int)((n + K2_KC - 1) / K2_KC);
    // the 12 plan fragments of 8 are dealt to the two plan halves alternately (wp = 0: fragments 0, 2, ..; wp = 1: 1, 3, ..), so that a
    // partly filled tile leaves both halves -- they sit on different SM sub-partitions, each with its own DMMA pipe -- the same work:
    // nb = this warp's live fragments.  Which warp computes a plan does not change the order its dot products are summed in.
    const int nfrag = min(12, (Bact - p0 + 7) >> 3);
    const int nb = (nfrag - wp + 1) >> 1;
    const bool warp_live = nb > 0;

    // loader: thread t copies 16-byte pieces (row = t/16 + 16 i, columns kk, kk+1) for i < NCP; pointers are set up once
    constexpr int NCP = ROWS * (K2_KC / 2) / NT;             // 14 / 16 / 20 for WJ = 1 / 2 / 4 (exact)
    static_assert(ROWS * (K2_KC / 2) % NT == 0, "loader tiling");
    const int kk = (tid % K2_TPR) * 2;
    const double* srcp[NCP];
    bool rowok[NCP];
#pragma unroll
    for (int i = 0; i < NCP; ++i) {
        const int row = tid / K2_TPR + K2_RPP * i;
        if (row < TJ) { const int64_t j = j0 + row; rowok[i] = j < n; srcp[i] = Sinv + (rowok[i] ? j : 0) * lds + kk; }
        else { const int p = p0 + row - TJ; rowok[i] = p < Bact; srcp[i] = rhs + (int64_t)(rowok[i] ? p : 0) * ldn + kk; }
    }
    const uint32_t dst0 = (uint32_t)__cvta_generic_to_shared(k2sm) + (uint32_t)(((tid / K2_TPR) * K2_LD + kk) * 8);
    auto load_chunk = [&](int c, int stage) {
        const int64_t k0 = (int64_t)c * K2_KC;
        const bool kok = k0 + kk < n;
        const uint32_t d = dst0 + (uint32_t)stage * (ROWS * K2_LD * 8);
#pragma unroll
        for (int i = 0; i < NCP; ++i) {
            const int sz = (kok && rowok[i]) ? 16 : 0;
            asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;" ::"r"(d + (uint32_t)(i * K2_RPP * K2_LD * 8)),
                         "l"(kok ? srcp[i] + k0 : srcp[i]), "r"(sz), "l"(tc::kEvictLast) : "memory");
        }
    };

    double acc[RA][6][2];
#pragma unroll
    for (int a = 0; a < RA; ++a)
#pragma unroll
        for (int b = 0; b < 6; ++b) { acc[a][b][0] = 0.0; acc[a][b][1] = 0.0; }

#pragma unroll
    for (int s = 0; s < K2_STAGES - 1; ++s) { if (s < nchunks) load_chunk(s, s); cp_async_commit(); }
    for (int c = 0; c < nchunks; ++c) {
        cp_async_wait<K2_STAGES - 2>();
        __syncthreads();
        if (c + K2_STAGES - 1 < nchunks) load_chunk(c + K2_STAGES - 1, (c + K2_STAGES - 1) % K2_STAGES);
        cp_async_commit();
        if (warp_live) {
            const double* sA = k2sm + (size_t)(c % K2_STAGES) * ROWS * K2_LD + (wj * RW + g) * K2_LD + q;
            const double* sB = k2sm + (size_t)(c % K2_STAGES) * ROWS * K2_LD + (TJ + wp * 8 + g) * K2_LD + q;
#pragma unroll
            for (int i = 0; i < K2_KC / 4 / KS; ++i) {
                const int ks = kq + i * KS;
                double av[RA];
#pragma unroll
                for (int a = 0; a < RA; ++a) av[a] = sA[a * 8 * K2_LD + ks * 4];
#pragma unroll
                for (int b = 0; b < 6; ++b) {
                    if (b < nb) {
                        const double bv = sB[b * 16 * K2_LD + ks * 4];
#pragma unroll
                        for (int a = 0; a < RA; ++a) dmma884(acc[a][b], av[a], bv);
                    }
                }
            }
        }
    }
    cp_async_wait<0>();
    __syncthreads();

    // ---- sum the k-slices in a fixed order: slices 1.. park their fragments, slice 0 adds them
    constexpr int FR = RA * 12;                            // accumulator doubles per thread
    double* red = k2sm;                                    // [(KS-1)][2 WJ warps][FR][32]
    constexpr size_t RED = (size_t)(KS - 1) * 2 * WJ * FR * 32;
    double* sacc = k2sm + (RED > (size_t)3 * 2 * 48 * 32 ? RED : (size_t)3 * 2 * 48 * 32);         // [2 WJ warps][48 plans][kNumResid]  (past the red area)
    if (KS > 1) {
        if (kq > 0) {
            double* dst = red + ((size_t)((kq - 1) * 2 * WJ + wp * WJ + wj) * FR) * 32 + lane;
#pragma unroll
            for (int a = 0; a < RA; ++a)
#pragma unroll
                for (int b = 0; b < 6; ++b) { dst[((a * 6 + b) * 2 + 0) * 32] = acc[a][b][0]; dst[((a * 6 + b) * 2 + 1) * 32] = acc[a][b][1]; }
        }
        __syncthreads();
        if (kq == 0) {
            for (int k = 1; k < KS; ++k) {
                const double* src = red + ((size_t)((k - 1) * 2 * WJ + wp * WJ + wj) * FR) * 32 + lane;
#pragma unroll
                for (int a = 0; a < RA; ++a)
#pragma unroll
                    for (int b = 0; b < 6; ++b) { acc[a][b][0] += src[((a * 6 + b) * 2 + 0) * 32]; acc[a][b][1] += src[((a * 6 + b) * 2 + 1) * 32]; }
            }
        }
    }
    const int ew = wp * WJ + wj;                           // index of this (kq == 0) warp among the 2 WJ epilogue warps

    // ---- epilogue-2: thread owns rows j = j0 + wj*RW + a*8 + g, plans p = p0 + (2b + wp)*8 + 2q + e
    const bool resid = resid_partial != nullptr;
    if (kq == 0) {
#pragma unroll
    for (int b = 0; b < 6; ++b) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int p = p0 + (2 * b + wp) * 8 + 2 * q + e;
            double ra[kNumResid] = {0, 0, 0, 0, 0};
            if (p < Bact) {
                const double bp = beta[p];
#pragma unroll
                for (int a = 0; a < RA; ++a) {
                    const int64_t j = j0 + wj * RW + a * 8 + g;
                    if (j >= n) continue;
                    const double bh = Rb[j] * bp;
                    const double s_old = s2[(int64_t)p * ldn + j];
                    const double z_old = fmin(s_old, bh);
                    const double v = acc[a][b][e];
                    const double s_new = z_old + v;                       // s2+ = x2+ + y2 = v + z2   (Eq. 7)
                    const double z_new = fmin(s_new, bh);                 // (4b)
                    s2[(int64_t)p * ldn + j] = s_new;
                    const double rv = R[j] * v;
                    emit_small(v_hi, v_lo, (int64_t)p * ldn, j, rv, bf16 != 0);
                    if (resid) {
                        const double y_old = s_old - z_old, y_new = s_new - z_new, x = s_new - y_old;
                        ra[0] += (x - z_new) * (x - z_new);
                        ra[1] += (z_new - z_old) * (z_new - z_old);
                        ra[2] += x * x; ra[3] += z_new * z_new; ra[4] += y_new * y_new;
                    }
                }
            }
            if (resid) {
                // the 8 lanes with the same q hold the 8 row groups: fixed-order butterfly over g
#pragma unroll
                for (int t = 0; t < kNumResid; ++t) {
                    double v = ra[t];
                    v += __shfl_xor_sync(0xffffffffu, v, 4);
                    v += __shfl_xor_sync(0xffffffffu, v, 8);
                    v += __shfl_xor_sync(0xffffffffu, v, 16);
                    if (g == 0) sacc[(ew * 48 + b * 8 + 2 * q + e) * kNumResid + t] = v;
                }
            }
        }
    }
    }
    if (resid) {
        __syncthreads();
        for (int i = tid; i < K2_TP * kNumResid; i += NT) {
            const int pp = i / kNumResid, t = i % kNumResid;     // pp in [0, 96): fragment pp / 8 = 2 b + wp
            if (p0 + pp >= Bact) continue;
            const int f = pp >> 3;
            double v = 0.0;
            for (int w = 0; w < WJ; ++w) v += sacc[((((f & 1) * WJ + w) * 48) + (f >> 1) * 8 + (pp & 7)) * kNumResid + t];
            resid_partial[((int64_t)blockIdx.x * kMaxBpad + p0 + pp) * kNumResid + t] = v;
        }
    }
}

// ------------------------------------------------------------------------------------------ stopping rule (R7) + compaction (H5)
// One warp per slot: the per-CTA partials of both blocks are summed in a fixed order (lane-strided, then a butterfly),
// so the decision is deterministic; then the Boyd test.  Also records, per PLAN, the iteration count and the residual norms of
// every live plan at this check (a plan that freezes now keeps these values).
__global__ void convergence_kernel(const float* __restrict__ r1, int grid1, const double* __restrict__ r2, int grid2,
                                   const int32_t* __restrict__ bact_dev, int Bact, double dim_sqrt, float tol, float eps_abs, int it,
                                   const int32_t* __restrict__ slot_plan, int32_t* __restrict__ flags,
                                   int32_t* __restrict__ iters_plan, float* __restrict__ res_plan) {
    const int p = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (bact_dev) Bact = min(Bact, *bact_dev);
    if (p >= Bact) return;
    double a[kNumResid] = {0, 0, 0, 0, 0};
    for (int g = lane; g < grid1; g += 32)
        for (int t = 0; t < kNumResid; ++t) a[t] += (double)r1[((int64_t)g * kMaxBpad + p) * kNumResid + t];
    for (int g = lane; g < grid2; g += 32)
        for (int t = 0; t < kNumResid; ++t) a[t] += r2[((int64_t)g * kMaxBpad + p) * kNumResid + t];
    for (int t = 0; t < kNumResid; ++t) a[t] = warp_sum(a[t]);
    if (lane != 0) return;
    const double rp = sqrt(a[0]), rd = sqrt(a[1]), nx = sqrt(a[2]), nz = sqrt(a[3]), ny = sqrt(a[4]);
    const bool ok = (rp <= (double)eps_abs * dim_sqrt + (double)tol * fmax(nx, nz)) &&
                    (rd <= (double)eps_abs * dim_sqrt + (double)tol * ny);
    flags[p] = (ok && tol > 0.f) ? 1 : 0;
    const int plan = slot_plan[p];
    iters_plan[plan] = it;
    res_plan[2 * plan] = (float)rp;
    res_plan[2 * plan + 1] = (float)rd;
}

// Compaction decided on the device (one thread: at most 496 slots, a few table entries each).  With L live plans left after
// this check, the live range becomes [0, L): every flagged slot below L (a hole) trades places with an unflagged slot at or above L
// (a mover), so a frozen plan keeps its state (the iterate that passed the test) behind the live range.  Holes and movers are all
// different slots, so the row moves (move_rows_kernel, from the list written here) are independent of one another.
__global__ void compact_kernel(int32_t* __restrict__ bact, const int32_t* __restrict__ flags, int32_t* __restrict__ slot_plan,
                               float* __restrict__ utab, float* __restrict__ crtab, double* __restrict__ beta,
                               double* __restrict__ rho, double* __restrict__ wnorm, int32_t* __restrict__ moves,
                               int32_t* __restrict__ nmoves) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int B = *bact;
    int live = 0, nm = 0;
    for (int s = 0; s < B; ++s) live += flags[s] ? 0 : 1;
    int mover = B - 1;
    for (int hole = 0; hole < live; ++hole) {
        if (!flags[hole]) continue;
        while (flags[mover]) --mover;                       // an unflagged slot >= live exists for every hole
        const int s = hole, last = mover;
        for (int k = 0; k < kMaxClasses; ++k) {
            float tu = utab[k * kMaxBpad + s]; utab[k * kMaxBpad + s] = utab[k * kMaxBpad + last]; utab[k * kMaxBpad + last] = tu;
            float tcr = crtab[k * kMaxBpad + s]; crtab[k * kMaxBpad + s] = crtab[k * kMaxBpad + last]; crtab[k * kMaxBpad + last] = tcr;
            double tw = wnorm[s * kMaxClasses + k]; wnorm[s * kMaxClasses + k] = wnorm[last * kMaxClasses + k]; wnorm[last * kMaxClasses + k] = tw;
        }
        double tb = beta[s]; beta[s] = beta[last]; beta[last] = tb;
        double tr = rho[s]; rho[s] = rho[last]; rho[last] = tr;
        int tp = slot_plan[s]; slot_plan[s] = slot_plan[last]; slot_plan[last] = tp;
        moves[2 * nm] = s; moves[2 * nm + 1] = last; ++nm;
        --mover;
    }
    *bact = live;
    *nmoves = nm;
}

// move m: frozen slot a (a hole) <-> live slot b (its mover).  s1 and s2 are swapped (the frozen state is an output); the K1 operand G only moves
// b -> a (a frozen plan needs no operand).  Rows are walked as 16-byte words; grid = (chunks, upper bound on the moves).
__global__ void move_rows_kernel(const int32_t* __restrict__ moves, const int32_t* __restrict__ nmoves, float4* __restrict__ s1,
                                 float4* __restrict__ ghi, float4* __restrict__ glo, int64_t ldN4, double2* __restrict__ s2, int64_t ldn2) {
    const int m = blockIdx.y;
    if (m >= *nmoves) return;
    const int a = moves[2 * m], b = moves[2 * m + 1];
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, t0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    float4* sa = s1 + (int64_t)a * ldN4; float4* sb = s1 + (int64_t)b * ldN4;
    float4* ha = ghi + (int64_t)a * ldN4; const float4* hb = ghi + (int64_t)b * ldN4;
    float4* la = glo + (int64_t)a * ldN4; const float4* lb = glo + (int64_t)b * ldN4;
    for (int64_t i = t0; i < ldN4; i += stride) {
        const float4 x = sa[i], y = sb[i];
        sa[i] = y; sb[i] = x;
        ha[i] = hb[i]; la[i] = lb[i];
    }
    double2* qa = s2 + (int64_t)a * ldn2; double2* qb = s2 + (int64_t)b * ldn2;
    for (int64_t i = t0; i < ldn2; i += stride) {
        const double2 x = qa[i], y = qb[i];
        qa[i] = y; qb[i] = x;
    }
}

// ------------------------------------------------------------------------------------------ presolve: the box optimum
// x_box = argmin c^T x over the box alone (x = u where c < 0, 0 where c > 0; Eq. 1).  If A x_box <= b it is optimal
// for the LP, t* = 0, and the ADMM fixed point is known in closed form: z1 = x_box, y1 = -c/rho, z2 = A x_box, y2 = 0 (Eq. 6-7 with
// v = y2 = 0).  presolve_state_kernel writes s1 = z1 + y1 of that candidate for every plan (emit_g then yields G = a o z1, and the K1
// contraction A^ z1); presolve_test_kernel accepts a plan iff A^ z1 <= b^ (1 - margin) in every row and then stores s2 = z2.
__global__ void presolve_state_kernel(const EpiParams ep, int B) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;
    if (i >= ep.N || p >= B) return;
    const int cls = ep.point_class[i];
    const float cr = ep.crtab[cls * kMaxBpad + p];
    const float ub = mask_ub(ep, cls, p, i);
    ep.s1[(int64_t)p * ep.ldN + i] = (cr < 0.f ? ub : 0.f) - cr;
}
// one block per plan.  flags: 1 = accepted (settled, 0 iterations); 0 = rejected, starts from the zero iterate (R6); 2 = rejected
// but warm-started (deviation D3): its box optimum violates A x <= b by at most a factor warm_ratio in every row, and the box
// state (z1 = x_box, y1 = -c/rho, z2 = min(A x_box, b), y2 = the excess) is kept as its initial iterate.
__global__ void presolve_test_kernel(const float* __restrict__ partial, const int32_t* __restrict__ mtile_slot_begin, int n_mma,
                                     const double* __restrict__ R, const double* __restrict__ Rb, const double* __restrict__ beta,
                                     int64_t n, int64_t ldn, int slot0, int nact, double margin, double warm_ratio,
                                     double* __restrict__ s2, int32_t* __restrict__ flags) {
    const int p = blockIdx.x;
    if (p >= nact) return;
    const int gs = slot0 + p;
    __shared__ int bad, cold;
    if (threadIdx.x == 0) { bad = 0; cold = 0; }
    __syncthreads();
    const double bp = beta[gs];
    int mybad = 0, mycold = 0;
    for (int64_t j = threadIdx.x; j < n; j += blockDim.x) {
        const int mt = (int)(j / kTileM), jl = (int)(j % kTileM);
        double w = 0.0;
        for (int s = mtile_slot_begin[mt]; s < mtile_slot_begin[mt + 1]; ++s)
            w += (double)partial[((int64_t)s * n_mma + p) * kTileM + jl];
        w *= R[j];
        const double bj = Rb[j] * bp;
        if (!(w <= bj * (1.0 - margin))) mybad = 1;
        if (!(w <= bj * warm_ratio)) mycold = 1;           // (A x_box)_j / b_j above the ratio (or b_j = 0 < (A x_box)_j)
        s2[(int64_t)gs * ldn + j] = w;                     // s2 = A x_box of the candidate; overwritten with 0 below for a cold start
    }
    if (mybad) bad = 1;
    if (mycold) cold = 1;
    __syncthreads();
    const int rejected = bad, warm = rejected && warm_ratio > 0.0 && !cold;
    if (rejected && !warm)
        for (int64_t j = threadIdx.x; j < n; j += blockDim.x) s2[(int64_t)gs * ldn + j] = 0.0;
    if (threadIdx.x == 0) flags[gs] = rejected ? (warm ? 2 : 0) : 1;
}
// zero start (R6) for the plans the presolve neither accepted nor warm-started; their K1 operand is re-emitted by emit_g afterwards
__global__ void presolve_reset_kernel(const int32_t* __restrict__ flags, float* __restrict__ s1, int64_t N, int64_t ldN, int B) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;
    if (i >= N || p >= B || flags[p]) return;
    s1[(int64_t)p * ldN + i] = 0.f;
}
// after the reset: only the accepted plans stay flagged (the compaction freezes every flagged slot)
__global__ void presolve_flags_kernel(int32_t* __restrict__ flags, int B) {
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < B) flags[p] = flags[p] == 1 ? 1 : 0;
}
__global__ void set_iters_kernel(const int32_t* __restrict__ flags, int B, int32_t* __restrict__ iters_plan, float* __restrict__ res_plan) {
    int p = blockIdx.x * blockDim.x + threadIdx.x;        // slot == plan before any compaction
    if (p >= B) return;
    iters_plan[p] = 0; res_plan[2 * p] = 0.f; res_plan[2 * p + 1] = 0.f;
    (void)flags;
}

// ------------------------------------------------------------------------------------------ SIMT cross-check contractions
// C[m][q] = sum_{k in [k0,k1)} X[m][k] * (Yhi[q][k] + Ylo[q][k]);  X [M][ldx], Y [Q][ldy]; 64x64 tile, 256 threads.
template <int EPI>
__global__ void __launch_bounds__(256) simt_contract_kernel(const float* __restrict__ X, int64_t M, int64_t ldx,
                                                            const float* __restrict__ Yhi, const float* __restrict__ Ylo,
                                                            int Q, int64_t ldy, int64_t K, int64_t k_per_split,
                                                            float* __restrict__ out, int64_t out_ld, int n_mma, int splits) {
    __shared__ float sX[16][64 + 1];
    __shared__ float sY[16][64 + 1];
    const int64_t m0 = (int64_t)blockIdx.x * 64;
    const int q0 = blockIdx.y * 64;
    const int split = blockIdx.z;
    const int64_t kbeg = (int64_t)split * k_per_split;
    const int64_t kend = (kbeg + k_per_split < K) ? kbeg + k_per_split : K;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float c[4][4] = {};
    for (int64_t k0 = kbeg; k0 < kend; k0 += 16) {
        for (int i = threadIdx.x; i < 16 * 64; i += 256) {
            int kk = i & 15, r = i >> 4;
            int64_t k = k0 + kk;
            int64_t m = m0 + r; int q = q0 + r;
            sX[kk][r] = (k < kend && m < M) ? X[m * ldx + k] : 0.f;
            sY[kk][r] = (k < kend && q < Q) ? (Yhi[(int64_t)q * ldy + k] + Ylo[(int64_t)q * ldy + k]) : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
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
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            int64_t m = m0 + ty * 4 + a; int q = q0 + tx * 4 + b;
            if (m >= M || q >= Q) continue;
            if (EPI == EPI_K1_PARTIAL) {
                // same layout as the tcgen05 path: partial[slot = mt * splits + split][q][m % 128]
                int64_t mt = m / kTileM;
                out[((mt * splits + split) * n_mma + q) * kTileM + (m % kTileM)] = c[a][b];
            } else {
                out[(int64_t)q * out_ld + m] = c[a][b];      // Q buffer [plan][point]
            }
        }
}

// epilogue-1 / objective over a Q buffer [plan][point] (SIMT path only); one block = 128 points, all plans
__global__ void __launch_bounds__(128) simt_epilogue_kernel(const EpiParams ep, int epi, const float* __restrict__ qbuf) {
    const int64_t row = (int64_t)blockIdx.x * 128 + threadIdx.x;
    const bool valid = row < ep.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __shared__ float sacc[4][8];
    int cls = valid ? ep.point_class[row] : 0;
    const bool resid = (epi == EPI_K3_STATE) && ep.resid_partial != nullptr;
    for (int pp = 0; pp < ep.n_slots_active; ++pp) {
        const int p = ep.slot0 + pp;
        float racc[kNumResid] = {0, 0, 0, 0, 0};
        float hinge = 0.f;
        if (valid) {
            float q = qbuf[(int64_t)pp * ep.ldN + row];
            float ub = mask_ub(ep, cls, p, row);
            if (epi == EPI_K3_STATE) {
                float cr = ep.crtab[cls * kMaxBpad + p];
                int64_t idx = (int64_t)p * ep.ldN + row;
                Epi1Out o = epi1_element(ep.s1[idx], q, ep.a_cls[cls], cr, ub, resid, racc);
                ep.s1[idx] = o.s_new; emit_small(ep.g_hi, ep.g_lo, (int64_t)p * ep.ldN, row, o.g, ep.small_bf16 != 0);
            } else {
                bool on = true;
                if (ep.mask) on = (ep.mask[(int64_t)ep.slot_plan[p] * ep.mask_words + (row >> 5)] >> (row & 31)) & 1u;
                hinge = on ? fmaxf(0.f, ep.sense[cls] * (ep.thr[cls] - q)) : 0.f;
            }
        }
        if (resid || epi == EPI_OBJECTIVE) {
            const int nt = resid ? kNumResid : kMaxClasses;
            for (int t = 0; t < nt; ++t) {
                float v = resid ? racc[t] : ((valid && cls == t) ? hinge : 0.f);
                v = warp_sum(v);
                if (lane == 0) sacc[warp][t] = v;
            }
            __syncthreads();
            if (threadIdx.x < nt) {
                float v = sacc[0][threadIdx.x] + sacc[1][threadIdx.x] + sacc[2][threadIdx.x] + sacc[3][threadIdx.x];
                if (resid) ep.resid_partial[((int64_t)blockIdx.x * kMaxBpad + p) * kNumResid + threadIdx.x] = v;
                else ep.hinge_partial[((int64_t)blockIdx.x * kMaxBpad + p) * kMaxClasses + threadIdx.x] = (double)v;
            }
            __syncthreads();
        }
    }
}


// obj[slot] = sum_k wnorm[slot][k] * sum_cta hinge[cta][slot][k] + beta[slot] * sum_j bot[j] t[slot][j]     (fp64)
__global__ void objective_reduce_kernel(const double* __restrict__ hinge, int grid, const double* __restrict__ wnorm,
                                        const double* __restrict__ beta, const double* __restrict__ bot, const float* __restrict__ t,
                                        int64_t n, int64_t ldn, int B, double* __restrict__ obj) {
    int p = blockIdx.x;
    if (p >= B) return;
    double acc = 0.0;
    for (int64_t j = threadIdx.x; j < n; j += blockDim.x) acc += bot[j] * (double)t[(int64_t)p * ldn + j];     // the rows that carry w_BOT
    acc *= beta[p];
    for (int i = threadIdx.x; i < grid * kMaxClasses; i += blockDim.x) {
        int g = i / kMaxClasses, k = i % kMaxClasses;
        acc += wnorm[p * kMaxClasses + k] * hinge[((int64_t)g * kMaxBpad + p) * kMaxClasses + k];
    }
    __shared__ double sh[8];
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) { double v = 0; for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += sh[w]; obj[p] = v; }
}

__global__ void split_small_kernel(const float* __restrict__ x, int64_t count, int64_t ld, void* __restrict__ hi, void* __restrict__ lo, int bf16) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) emit_small(hi, lo, (i / ld) * ld, i % ld, x[i], bf16 != 0);
}
// out[p][j] = sum over the slots of j's m-tile of partial[slot][p][j % 128]   (test hook, fp64)
__global__ void reduce_partial_kernel(const float* __restrict__ partial, const int32_t* __restrict__ mtile_slot_begin, int n_mma,
                                      int64_t n, int nact, double* __restrict__ out) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;
    if (j >= n || p >= nact) return;
    int mt = (int)(j / kTileM), jl = (int)(j % kTileM);
    double w = 0.0;
    for (int s = mtile_slot_begin[mt]; s < mtile_slot_begin[mt + 1]; ++s)
        w += (double)partial[((int64_t)s * n_mma + p) * kTileM + jl];
    out[(int64_t)p * n + j] = w;
}

// Second-pass low-dose volumes (PAPER.md II.C.1, :110-114): bit i of in_vol[p] is set iff lo <= dose[p][i] < hi (fp32 compares);
// bit i of any_vol is set iff some plan has it.  One warp per 32 points and plan: the ballot IS the packed word.
__global__ void lowdose_volume_kernel(const float* __restrict__ dose, int64_t ld, int64_t N, int B, float lo, float hi,
                                      uint32_t* __restrict__ in_vol, int64_t words, uint32_t* __restrict__ any_vol) {
    const int64_t wd = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int p = blockIdx.y;
    if (wd >= words || p >= B) return;
    const int64_t i = wd * 32 + (threadIdx.x & 31);
    const float d = i < N ? dose[(int64_t)p * ld + i] : -1.0f;
    const bool in = i < N && d >= lo && d < hi;
    const uint32_t bits = __ballot_sync(0xffffffffu, in);
    if ((threadIdx.x & 31) == 0) {
        in_vol[(int64_t)p * words + wd] = bits;
        if (bits) atomicOr(any_vol + wd, bits);
    }
}

// dst[plan][j] = src[plan_slot[plan]][j]
__global__ void gather_rows_kernel(const float* __restrict__ src, int64_t ld, const int32_t* __restrict__ plan_slot, int B,
                                   int64_t n, float* __restrict__ dst) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;
    if (j < n && p < B) dst[(int64_t)p * n + j] = src[(int64_t)plan_slot[p] * ld + j];
}

}  // namespace

// ============================================================================================ host launchers
void launch_transpose(const float* src, int64_t rows, int64_t cols, int64_t ld_src, float* dst, int64_t ld_dst, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(cols, 32), (unsigned)cdiv(rows, 32));
    transpose_kernel<<<grid, dim3(32, 8), 0, s>>>(src, rows, cols, ld_src, dst, ld_dst);
}
void launch_pack_tiles(const float* src, int64_t src_rows, int64_t src_cols, int64_t ld_src, bool transpose, float* dst,
                       cudaStream_t s) {
    if (!transpose) {
        const int64_t KB = cdiv(src_cols, kBlockK), RT = cdiv(src_rows, kTileM);
        pack_tiles_kernel<false><<<dim3((unsigned)KB, (unsigned)RT), 256, 0, s>>>(src, src_rows, src_cols, ld_src, dst, KB);
    } else {
        const int64_t KB = cdiv(src_rows, kBlockK), RT = cdiv(src_cols, kTileM);
        pack_tiles_kernel<true><<<dim3((unsigned)KB, (unsigned)RT), 256, 0, s>>>(src, src_rows, src_cols, ld_src, dst, KB);
    }
}
void launch_pack_tiles_bf16(const float* src, int64_t src_rows, int64_t src_cols, int64_t ld_src, bool transpose, void* dst,
                            cudaStream_t s) {
    __nv_bfloat16* d = reinterpret_cast<__nv_bfloat16*>(dst);
    if (!transpose) {
        const int64_t KB = cdiv(src_cols, 64), RT = cdiv(src_rows, kTileM);
        pack_tiles_bf16_kernel<false><<<dim3((unsigned)KB, (unsigned)RT), 256, 0, s>>>(src, src_rows, src_cols, ld_src, d, KB);
    } else {
        const int64_t KB = cdiv(src_rows, 64), RT = cdiv(src_cols, kTileM);
        pack_tiles_bf16_kernel<true><<<dim3((unsigned)KB, (unsigned)RT), 256, 0, s>>>(src, src_rows, src_cols, ld_src, d, KB);
    }
}
void launch_round_bf16(float* x, int64_t count, cudaStream_t s) {
    round_bf16_kernel<<<(unsigned)cdiv(count, 256), 256, 0, s>>>(x, count);
}
void launch_scale_rows_to_f64(const float* phi, int64_t ld, int64_t row0, int64_t rows, int64_t n, const uint8_t* cls,
                              const double* a_cls, double* out, cudaStream_t s) {
    scale_rows_kernel<<<(unsigned)cdiv(rows * n, 256), 256, 0, s>>>(phi, ld, row0, rows, n, cls, a_cls, out);
}
void launch_round_tf32(float* x, int64_t count, cudaStream_t s) {
    round_tf32_kernel<<<(unsigned)cdiv(count, 256), 256, 0, s>>>(x, count);
}
void launch_finish_S(double* M, int64_t n, double* R, cudaStream_t s) {
    // M arrives with its LOWER triangle (column-major) == UPPER triangle (row-major) filled by the SYRK
    symmetrize_kernel<<<(unsigned)cdiv(n * n, 256), 256, 0, s>>>(M, n, 0);
    make_R_kernel<<<(unsigned)cdiv(n, 256), 256, 0, s>>>(M, n, R);
    finish_S_kernel<<<(unsigned)cdiv(n * n, 256), 256, 0, s>>>(M, n, R);
}
void launch_symmetrize(double* A, int64_t n, cudaStream_t s) {
    symmetrize_kernel<<<(unsigned)cdiv(n * n, 256), 256, 0, s>>>(A, n, 0);
}
void launch_count_active(const uint32_t* mask, int64_t mask_words, const uint8_t* cls, int64_t N, int B, int32_t* counts,
                         cudaStream_t s) {
    count_active_kernel<<<B, 256, 0, s>>>(mask, mask_words, cls, N, counts);
}
void launch_emit_g(const EpiParams& ep, int Bact, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(ep.N, 256), Bact);
    emit_g_kernel<<<grid, 256, 0, s>>>(ep, Bact);
}
void launch_k2a(admm_handle* h, int slot0, int nact, int n_mma, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(h->n, 128), nact);
    k2a_kernel<<<grid, 128, 0, s>>>(h->d_partial, h->d_mtile_slot_begin, n_mma, h->d_s2, h->d_R, h->d_Rb, h->d_beta, h->n, h->ldn,
                                    slot0, nact, h->d_bact, h->d_rhs);
    h->launch_count++;
}
// Rows of the K2b block tile: 16, 32, 40, 48 or 64.  One block per SM fits (its cp.async ring takes ~140-200 KB), so the launch runs
// in waves of sm_count blocks and the last, partly filled wave costs a full one: n = 9600 is 300 tiles of 32 rows = 3 waves for 148
// SMs, but 240 tiles of 40 rows = 2.  Measured on B200 (96 plans; microseconds per wave per 9600 columns): 215 / 338 / 438 / 511 / 597
// for 16 / 32 / 40 / 48 / 64 rows = the relative block costs below; K2a + K2b at n = 9600: 1073 / 1015 / 876 / 1022 / 1194 us, at
// n = 12000: 1586 / 1260 / 1592 / 1244 / 1485 us.  The choice minimises waves x cost and depends on n ONLY: the summation order of a
// row's dot product depends on the tile (its k-slices), and a plan must come out bit-identical whatever the batch it is solved in.
int k2_choose_rows(const admm_handle* h, int) {
#ifdef K2_FORCE_ROWS          // compile-time override, for measuring one tile against another (nvcc -DK2_FORCE_ROWS=32)
    return K2_FORCE_ROWS;
#endif
    const int rows[5] = {16, 32, 40, 48, 64};
    const double cost[5] = {0.36, 0.57, 0.72, 0.84, 1.0};
    int best = 16; double best_t = 1e300;
    for (int i = 0; i < 5; ++i) {
        const double t = (double)cdiv(cdiv(h->n, rows[i]), h->sm_count) * cost[i];
        if (t <= best_t * (1.0 + 1e-9)) { best_t = std::min(t, best_t); best = rows[i]; }      // ties go to the larger tile
    }
    return best;
}
int k2b_grid(const admm_handle* h, int) { return (int)cdiv(h->n, h->k2_rows); }
template <int WJ, int RA>
static void launch_k2b_t(admm_handle* h, int Bact, bool resid, cudaStream_t s) {
    constexpr int TJ = 8 * RA * WJ;
    const size_t smem = (size_t)k2_stages(TJ) * (TJ + K2_TP) * K2_LD * sizeof(double);
    // the attribute is per device: set it per handle and instantiation (a process-wide flag would leave a second device without the opt-in)
    if (h->k2_attr_tj != TJ) { cudaFuncSetAttribute(k2b_kernel<WJ, RA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); h->k2_attr_tj = TJ; }
    dim3 grid((unsigned)cdiv(h->n, TJ), (unsigned)cdiv(Bact, K2_TP));
    k2b_kernel<WJ, RA><<<grid, 256, smem, s>>>(h->d_Sinv, h->lds, h->d_rhs, h->d_s2, h->d_R, h->d_Rb, h->d_beta, h->n, h->ldn, Bact, h->d_bact,
                                               h->d_vhi, h->d_vlo, h->opt.storage == ADMM_STORAGE_BF16 ? 1 : 0,
                                               resid ? h->d_resid2 : nullptr);
}
void launch_k2b(admm_handle* h, int Bact, bool resid, cudaStream_t s) {
    switch (h->k2_rows) {                     // <row groups WJ, 8-row fragments per warp RA>: block tile = 8 RA WJ rows
        case 64: launch_k2b_t<4, 2>(h, Bact, resid, s); break;      // (a 32 x 48 warp tile, <2, 4>, measured slower: 1.42 vs 1.33 ms at config 2)
        case 48: launch_k2b_t<1, 6>(h, Bact, resid, s); break;
        case 40: launch_k2b_t<1, 5>(h, Bact, resid, s); break;
        case 32: launch_k2b_t<2, 2>(h, Bact, resid, s); break;
        default: launch_k2b_t<1, 2>(h, Bact, resid, s); break;
    }
    h->launch_count++;
}
void launch_simt_k1(admm_handle* h, int slot0, int nact, int n_mma, int splits, cudaStream_t s) {
    if (h->opt.storage == ADMM_STORAGE_CSR) { launch_csr_k1(h, slot0, nact, n_mma, s); return; }
    const int64_t k_per_split = cdiv(cdiv(h->N, splits), 16) * 16;
    dim3 grid((unsigned)cdiv(h->n, 64), (unsigned)cdiv(nact, 64), splits);
    simt_contract_kernel<EPI_K1_PARTIAL><<<grid, 256, 0, s>>>(h->d_phiT, h->n, h->ldN, h->d_ghi + (int64_t)slot0 * h->ldN,
                                                               h->d_glo + (int64_t)slot0 * h->ldN, nact, h->ldN, h->N,
                                                               k_per_split, h->d_partial, 0, n_mma, splits);
    h->launch_count++;
}
void launch_simt_k3(admm_handle* h, const EpiParams& ep, int epi, const float* vhi, const float* vlo, float* qbuf,
                    cudaStream_t s) {
    // vhi / vlo point at the first slot of this pass
    const int nact = ep.n_slots_active;
    if (h->opt.storage == ADMM_STORAGE_CSR) {
        launch_csr_k3(h, nact, vhi, vlo, qbuf, s);
        simt_epilogue_kernel<<<(unsigned)cdiv(h->N, 128), 128, 0, s>>>(ep, epi, qbuf);
        h->launch_count += 1;
        return;
    }
    dim3 grid((unsigned)cdiv(h->N, 64), (unsigned)cdiv(nact, 64), 1);
    simt_contract_kernel<EPI_K3_STATE><<<grid, 256, 0, s>>>(h->d_phi, h->N, h->ldn, vhi, vlo, nact, h->ldn, h->n, h->n,
                                                             qbuf, h->ldN, 0, 1);
    simt_epilogue_kernel<<<(unsigned)cdiv(h->N, 128), 128, 0, s>>>(ep, epi, qbuf);
    h->launch_count += 2;
}
void launch_convergence(admm_handle* h, int Bact, int grid1, int grid2, float tol, float eps_abs, int it, cudaStream_t s) {
    convergence_kernel<<<(unsigned)cdiv(Bact, 4), 128, 0, s>>>(h->d_resid1, grid1, h->d_resid2, grid2, h->d_bact, Bact,
                                                              sqrt((double)(h->N + h->n)), tol, eps_abs, it, h->d_slot_plan,
                                                              h->d_conv_flags, h->d_iters_plan, h->d_res_plan);
    h->launch_count++;
}
// H5 on the device: shrink the live range, fix the per-slot tables, move the rows.  `Bact` is the host's upper bound on the live count.
void launch_compaction(admm_handle* h, int Bact, cudaStream_t s) {
    compact_kernel<<<1, 32, 0, s>>>(h->d_bact, h->d_conv_flags, h->d_slot_plan, h->d_utab, h->d_crtab, h->d_beta, h->d_rho,
                                    h->d_wnorm, h->d_moves, h->d_nmoves);
    const int64_t ldN4 = h->ldN / 4, ldn2 = h->ldn / 2;
    const unsigned gx = (unsigned)std::max<int64_t>(1, std::min<int64_t>(64, cdiv(ldN4, 256)));
    move_rows_kernel<<<dim3(gx, (unsigned)std::max(1, Bact / 2)), 256, 0, s>>>(
        h->d_moves, h->d_nmoves, reinterpret_cast<float4*>(h->d_s1), reinterpret_cast<float4*>(h->d_ghi),
        reinterpret_cast<float4*>(h->d_glo), ldN4, reinterpret_cast<double2*>(h->d_s2), ldn2);
    h->launch_count += 2;
}
void launch_presolve_state(const EpiParams& ep, int B, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(ep.N, 256), B);
    presolve_state_kernel<<<grid, 256, 0, s>>>(ep, B);
}
void launch_presolve_test(admm_handle* h, int slot0, int nact, int n_mma, double margin, cudaStream_t s) {
    presolve_test_kernel<<<nact, 256, 0, s>>>(h->d_partial, h->d_mtile_slot_begin, n_mma, h->d_R, h->d_Rb, h->d_beta, h->n, h->ldn, slot0, nact,
                                               margin, (double)h->opt.warm_start_ratio, h->d_s2, h->d_conv_flags);
}
void launch_presolve_reset(admm_handle* h, int B, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(h->N, 256), B);
    presolve_reset_kernel<<<grid, 256, 0, s>>>(h->d_conv_flags, h->d_s1, h->N, h->ldN, B);
    presolve_flags_kernel<<<(unsigned)cdiv(B, 128), 128, 0, s>>>(h->d_conv_flags, B);
}
void launch_init_plan_records(admm_handle* h, int B, cudaStream_t s) {
    set_iters_kernel<<<(unsigned)cdiv(B, 128), 128, 0, s>>>(h->d_conv_flags, B, h->d_iters_plan, h->d_res_plan);
}
void launch_make_t(admm_handle* h, int Bact, void* t_hi, void* t_lo, float* t_f32, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(h->n, 128), Bact);
    make_t_kernel<<<grid, 128, 0, s>>>(h->d_s2, h->d_R, h->d_Rb, h->d_beta, h->d_rho, h->n, h->ldn, Bact, t_hi, t_lo, t_f32,
                                       h->opt.storage == ADMM_STORAGE_BF16 ? 1 : 0);
    h->launch_count++;
}
void launch_split_small(const float* x, int64_t count, int64_t ld, void* hi, void* lo, bool bf16, cudaStream_t s) {
    split_small_kernel<<<(unsigned)cdiv(count, 256), 256, 0, s>>>(x, count, ld, hi, lo, bf16 ? 1 : 0);
}
void launch_reduce_partial(admm_handle* h, int nact, int n_mma, double* out, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(h->n, 128), nact);
    reduce_partial_kernel<<<grid, 128, 0, s>>>(h->d_partial, h->d_mtile_slot_begin, n_mma, h->n, nact, out);
}
void launch_objective_reduce(admm_handle* h, int B, int grid, const float* t_f32, const double* wnorm, double* obj_slot,
                             cudaStream_t s) {
    objective_reduce_kernel<<<B, 256, 0, s>>>(h->d_hinge, grid, wnorm, h->d_beta, h->d_bot, t_f32, h->n, h->ldn, B, obj_slot);
    h->launch_count++;
}
void launch_lowdose_volume(const float* dose, int64_t ld, int64_t N, int B, float lo, float hi, uint32_t* in_vol, int64_t words,
                           uint32_t* any_vol, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(words, 8), (unsigned)B);
    lowdose_volume_kernel<<<grid, 256, 0, s>>>(dose, ld, N, B, lo, hi, in_vol, words, any_vol);
}
void launch_gather_rows(const float* src, int64_t ld, const int32_t* plan_slot, int B, int64_t n, float* dst, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(n, 256), B);
    gather_rows_kernel<<<grid, 256, 0, s>>>(src, ld, plan_slot, B, n, dst);
}
void launch_state_out(admm_handle* h, const EpiParams& ep, int slot, float* z1, float* y1, double* z2,
                      double* y2, cudaStream_t s) {
    int64_t m = h->N > h->n ? h->N : h->n;
    state_out_kernel<<<(unsigned)cdiv(m, 256), 256, 0, s>>>(ep, slot, h->d_s2, h->d_Rb, h->d_beta, z1, y1, z2, y2);     // Rb: the bound b_hat = Rb w_BOT
}
