// Everything on the hot path that is not a tcgen05 contraction: the S^-1 apply with fused epilogue-2
// (K2a/K2b), the stopping rule, state start-up / read-out, setup helpers, and the plain-FFMA
// cross-check versions of K1/K3 (ADMM_PATH_SIMT).
#include <cstdio>
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
    float hi = tc::tf32_rn(g);
    ep.g_hi[(int64_t)p * ep.ldN + i] = hi;
    ep.g_lo[(int64_t)p * ep.ldN + i] = g - hi;
}

__global__ void state_out_kernel(const EpiParams ep, int slot, const double* __restrict__ s2, const double* __restrict__ R,
                                 double beta, float* z1, float* y1, double* z2, double* y2) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
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
__global__ void make_t_kernel(const double* __restrict__ s2, const double* __restrict__ R, const double* __restrict__ beta,
                              const double* __restrict__ rho, int64_t n, int64_t ldn, int Bact,
                              float* __restrict__ t_hi, float* __restrict__ t_lo, float* __restrict__ t_f32) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;
    if (j >= n || p >= Bact) return;
    double y2 = fmax(s2[(int64_t)p * ldn + j] - R[j] * beta[p], 0.0);
    double t = rho[p] * R[j] * y2;
    float tf = (float)t;
    float hi = tc::tf32_rn(tf);
    t_hi[(int64_t)p * ldn + j] = hi;
    t_lo[(int64_t)p * ldn + j] = tc::tf32_rn((float)(t - (double)hi));
    t_f32[(int64_t)p * ldn + j] = tf;
}

// ------------------------------------------------------------------------------------------ K2a: rhs of Eq. (6)
// rhs[p][j] = R_j * sum_slots partial[slot][p][j - 128 mt]  -  (2 z2 - s2)[p][j]     (fp64)
__global__ void k2a_kernel(const float* __restrict__ partial, const int32_t* __restrict__ mtile_slot_begin, int n_mma,
                           const double* __restrict__ s2, const double* __restrict__ R, const double* __restrict__ beta,
                           int64_t n, int64_t ldn, int slot0, int nact, double* __restrict__ rhs) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;                       // index inside this contraction pass
    if (j >= n || p >= nact) return;
    int mt = (int)(j / kTileM), jl = (int)(j % kTileM);
    double w = 0.0;
    for (int s = mtile_slot_begin[mt]; s < mtile_slot_begin[mt + 1]; ++s)
        w += (double)partial[((int64_t)s * n_mma + p) * kTileM + jl];
    const int gs = slot0 + p;
    double sv = s2[(int64_t)gs * ldn + j];
    double z = fmin(sv, R[j] * beta[gs]);
    rhs[(int64_t)gs * ldn + j] = R[j] * w - (2.0 * z - sv);
}

// ------------------------------------------------------------------------------------------ K2b: v = S^-1 rhs + epilogue-2
// Tile: 32 plans x 32 columns per block of 128 threads (each thread 2 plans x 4 columns), k-chunks of 16.
// Epilogue (4b)/(4c) on block 2 in single-state form: s2+ = z2 + v, z2 = min(s2, R beta); emits V = R o v (tf32 hi/lo).
constexpr int K2_TP = 32, K2_TJ = 32, K2_TK = 16;
__global__ void __launch_bounds__(128) k2b_kernel(const double* __restrict__ Sinv, const double* __restrict__ rhs,
                                                  double* __restrict__ s2, const double* __restrict__ R,
                                                  const double* __restrict__ beta, int64_t n, int64_t ldn, int Bact,
                                                  float* __restrict__ v_hi, float* __restrict__ v_lo,
                                                  double* __restrict__ resid_partial) {
    __shared__ double sR[K2_TK][K2_TP + 1];     // rhs chunk, [k][p]
    __shared__ double sS[K2_TK][K2_TJ];         // Sinv chunk, [k][j]
    __shared__ double sacc[K2_TP][kNumResid];
    const int tx = threadIdx.x & 7;             // column group (4 columns)
    const int ty = threadIdx.x >> 3;            // plan group (2 plans)
    const int64_t j0 = (int64_t)blockIdx.x * K2_TJ;
    const int p0 = blockIdx.y * K2_TP;
    double c[2][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}};
    for (int64_t k0 = 0; k0 < n; k0 += K2_TK) {
        for (int i = threadIdx.x; i < K2_TK * K2_TP; i += 128) {
            int kk = i % K2_TK, pp = i / K2_TK;
            int64_t k = k0 + kk; int p = p0 + pp;
            sR[kk][pp] = (k < n && p < Bact) ? rhs[(int64_t)p * ldn + k] : 0.0;
        }
        for (int i = threadIdx.x; i < K2_TK * K2_TJ; i += 128) {
            int jj = i % K2_TJ, kk = i / K2_TJ;
            int64_t k = k0 + kk, j = j0 + jj;
            sS[kk][jj] = (k < n && j < n) ? Sinv[k * n + j] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < K2_TK; ++kk) {
            double r0 = sR[kk][ty * 2], r1 = sR[kk][ty * 2 + 1];
            double s0 = sS[kk][tx * 4], s1 = sS[kk][tx * 4 + 1], s2v = sS[kk][tx * 4 + 2], s3 = sS[kk][tx * 4 + 3];
            c[0][0] += r0 * s0; c[0][1] += r0 * s1; c[0][2] += r0 * s2v; c[0][3] += r0 * s3;
            c[1][0] += r1 * s0; c[1][1] += r1 * s1; c[1][2] += r1 * s2v; c[1][3] += r1 * s3;
        }
        __syncthreads();
    }
    const bool resid = resid_partial != nullptr;
    if (resid) {
        for (int i = threadIdx.x; i < K2_TP * kNumResid; i += 128) sacc[i / kNumResid][i % kNumResid] = 0.0;
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < 2; ++a) {
        const int p = p0 + ty * 2 + a;
        double acc[kNumResid] = {0, 0, 0, 0, 0};
        if (p < Bact) {
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const int64_t j = j0 + tx * 4 + b;
                if (j >= n) continue;
                const double bh = R[j] * beta[p];
                const double s_old = s2[(int64_t)p * ldn + j];
                const double z_old = fmin(s_old, bh);
                const double v = c[a][b];
                const double s_new = z_old + v;                       // s2+ = x2+ + y2 = v + z2   (Eq. 7)
                const double z_new = fmin(s_new, bh);                 // (4b)
                s2[(int64_t)p * ldn + j] = s_new;
                const double rv = R[j] * v;
                const float hi = tc::tf32_rn((float)rv);
                v_hi[(int64_t)p * ldn + j] = hi;
                v_lo[(int64_t)p * ldn + j] = tc::tf32_rn((float)(rv - (double)hi));
                if (resid) {
                    const double y_old = s_old - z_old, y_new = s_new - z_new, x = s_new - y_old;
                    acc[0] += (x - z_new) * (x - z_new);
                    acc[1] += (z_new - z_old) * (z_new - z_old);
                    acc[2] += x * x; acc[3] += z_new * z_new; acc[4] += y_new * y_new;
                }
            }
        }
        if (resid) {
            // the 8 threads with the same ty are consecutive lanes: reduce over tx with shuffles
#pragma unroll
            for (int t = 0; t < kNumResid; ++t) {
                double v = acc[t];
                v += __shfl_xor_sync(0xffffffffu, v, 1);
                v += __shfl_xor_sync(0xffffffffu, v, 2);
                v += __shfl_xor_sync(0xffffffffu, v, 4);
                if (tx == 0) sacc[ty * 2 + a][t] = v;
            }
        }
    }
    if (resid) {
        __syncthreads();
        for (int i = threadIdx.x; i < K2_TP * kNumResid; i += 128) {
            int pp = i / kNumResid, t = i % kNumResid;
            if (p0 + pp < Bact)
                resid_partial[((int64_t)blockIdx.x * kMaxBpad + p0 + pp) * kNumResid + t] = sacc[pp][t];
        }
    }
}

// ------------------------------------------------------------------------------------------ stopping rule (R7)
// One thread per slot: fixed-order sum of the per-CTA partials of both blocks, then the Boyd test.
__global__ void convergence_kernel(const float* __restrict__ r1, int grid1, const double* __restrict__ r2, int grid2,
                                   int Bact, double dim_sqrt, float tol, float eps_abs,
                                   int32_t* __restrict__ flags, float* __restrict__ res_slot) {
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= Bact) return;
    double a[kNumResid] = {0, 0, 0, 0, 0};
    for (int g = 0; g < grid1; ++g)
        for (int t = 0; t < kNumResid; ++t) a[t] += (double)r1[((int64_t)g * kMaxBpad + p) * kNumResid + t];
    for (int g = 0; g < grid2; ++g)
        for (int t = 0; t < kNumResid; ++t) a[t] += r2[((int64_t)g * kMaxBpad + p) * kNumResid + t];
    const double rp = sqrt(a[0]), rd = sqrt(a[1]), nx = sqrt(a[2]), nz = sqrt(a[3]), ny = sqrt(a[4]);
    const bool ok = (rp <= (double)eps_abs * dim_sqrt + (double)tol * fmax(nx, nz)) &&
                    (rd <= (double)eps_abs * dim_sqrt + (double)tol * ny);
    flags[p] = ok ? 1 : 0;
    res_slot[2 * p] = (float)rp;
    res_slot[2 * p + 1] = (float)rd;
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
                ep.s1[idx] = o.s_new; ep.g_hi[idx] = o.g_hi; ep.g_lo[idx] = o.g_lo;
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


// obj[slot] = sum_k wnorm[slot][k] * sum_cta hinge[cta][slot][k] + beta[slot] * sum_j t[slot][j]     (fp64)
__global__ void objective_reduce_kernel(const double* __restrict__ hinge, int grid, const double* __restrict__ wnorm,
                                        const double* __restrict__ beta, const float* __restrict__ t, int64_t n, int64_t ldn,
                                        int B, double* __restrict__ obj) {
    int p = blockIdx.x;
    if (p >= B) return;
    double acc = 0.0;
    for (int64_t j = threadIdx.x; j < n; j += blockDim.x) acc += (double)t[(int64_t)p * ldn + j];
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

__global__ void split_tf32_kernel(const float* __restrict__ x, int64_t count, float* __restrict__ hi, float* __restrict__ lo) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) { float h = tc::tf32_rn(x[i]); hi[i] = h; lo[i] = x[i] - h; }
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
    k2a_kernel<<<grid, 128, 0, s>>>(h->d_partial, h->d_mtile_slot_begin, n_mma, h->d_s2, h->d_R, h->d_beta, h->n, h->ldn,
                                    slot0, nact, h->d_rhs);
    h->launch_count++;
}
int k2b_grid(const admm_handle* h, int) { return (int)cdiv(h->n, K2_TJ); }
void launch_k2b(admm_handle* h, int Bact, bool resid, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(h->n, K2_TJ), (unsigned)cdiv(Bact, K2_TP));
    k2b_kernel<<<grid, 128, 0, s>>>(h->d_Sinv, h->d_rhs, h->d_s2, h->d_R, h->d_beta, h->n, h->ldn, Bact, h->d_vhi,
                                    h->d_vlo, resid ? h->d_resid2 : nullptr);
    h->launch_count++;
}
void launch_simt_k1(admm_handle* h, int slot0, int nact, int n_mma, int splits, cudaStream_t s) {
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
    dim3 grid((unsigned)cdiv(h->N, 64), (unsigned)cdiv(nact, 64), 1);
    simt_contract_kernel<EPI_K3_STATE><<<grid, 256, 0, s>>>(h->d_phi, h->N, h->ldn, vhi, vlo, nact, h->ldn, h->n, h->n,
                                                             qbuf, h->ldN, 0, 1);
    simt_epilogue_kernel<<<(unsigned)cdiv(h->N, 128), 128, 0, s>>>(ep, epi, qbuf);
    h->launch_count += 2;
}
void launch_convergence(admm_handle* h, int Bact, int grid1, int grid2, float tol, float eps_abs, cudaStream_t s) {
    convergence_kernel<<<(unsigned)cdiv(Bact, 64), 64, 0, s>>>(h->d_resid1, grid1, h->d_resid2, grid2, Bact,
                                                              sqrt((double)(h->N + h->n)), tol, eps_abs, h->d_conv_flags,
                                                              h->d_res_slot);
    h->launch_count++;
}
void launch_make_t(admm_handle* h, int Bact, float* t_hi, float* t_lo, float* t_f32, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(h->n, 128), Bact);
    make_t_kernel<<<grid, 128, 0, s>>>(h->d_s2, h->d_R, h->d_beta, h->d_rho, h->n, h->ldn, Bact, t_hi, t_lo, t_f32);
    h->launch_count++;
}
void launch_split_tf32(const float* x, int64_t count, float* hi, float* lo, cudaStream_t s) {
    split_tf32_kernel<<<(unsigned)cdiv(count, 256), 256, 0, s>>>(x, count, hi, lo);
}
void launch_reduce_partial(admm_handle* h, int nact, int n_mma, double* out, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(h->n, 128), nact);
    reduce_partial_kernel<<<grid, 128, 0, s>>>(h->d_partial, h->d_mtile_slot_begin, n_mma, h->n, nact, out);
}
void launch_objective_reduce(admm_handle* h, int B, int grid, const float* t_f32, const double* wnorm, double* obj_slot,
                             cudaStream_t s) {
    objective_reduce_kernel<<<B, 256, 0, s>>>(h->d_hinge, grid, wnorm, h->d_beta, t_f32, h->n, h->ldn, B, obj_slot);
    h->launch_count++;
}
void launch_gather_rows(const float* src, int64_t ld, const int32_t* plan_slot, int B, int64_t n, float* dst, cudaStream_t s) {
    dim3 grid((unsigned)cdiv(n, 256), B);
    gather_rows_kernel<<<grid, 256, 0, s>>>(src, ld, plan_slot, B, n, dst);
}
void launch_state_out(admm_handle* h, const EpiParams& ep, int slot, double beta, float* z1, float* y1, double* z2,
                      double* y2, cudaStream_t s) {
    int64_t m = h->N > h->n ? h->N : h->n;
    state_out_kernel<<<(unsigned)cdiv(m, 256), 256, 0, s>>>(ep, slot, h->d_s2, h->d_R, beta, z1, y1, z2, y2);
}
