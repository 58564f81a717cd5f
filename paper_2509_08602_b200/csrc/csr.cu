// ADMM_STORAGE_CSR (BASELINE.json config 4, last variant): Phi thresholded at csr_rel_threshold * max|Phi| and kept as
// CSR (rows = dose points, for Q = Phi V) plus the CSR of Phi^T (rows = time variables, for W = Phi^T G).
// The two contractions of Eq. (6)/(7) become SpMMs on the plain FP32 ALUs; everything else of the
// iteration (K2a/K2b, epilogue-1, stopping rule) is the code of the dense path.  S is formed from the THRESHOLDED
// matrix (api.cu zeroes the dropped entries before the SYRK), so the GPU solves exactly the LP of the thresholded Phi.
#include <cub/device/device_scan.cuh>

#include "admm_internal.h"
#include "epilogue.cuh"

namespace {

inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

__global__ void absmax_kernel(const float* __restrict__ x, int64_t count, unsigned int* __restrict__ out) {
    float m = 0.f;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x)
        m = fmaxf(m, fabsf(x[i]));
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));      // non-negative floats order like their bit patterns
}

__global__ void threshold_kernel(float* __restrict__ x, int64_t count, float tau) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count && fabsf(x[i]) < tau) x[i] = 0.f;
}

// one warp per row: number of non-zeros
__global__ void row_count_kernel(const float* __restrict__ X, int64_t rows, int64_t cols, int64_t ld, int64_t* __restrict__ cnt) {
    const int64_t r = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (r >= rows) return;
    int c = 0;
    for (int64_t j = lane; j < cols; j += 32) c += X[r * ld + j] != 0.f;
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) cnt[r] = c;
}

// one warp per row: ballot compaction keeps the columns in increasing order
__global__ void row_fill_kernel(const float* __restrict__ X, int64_t rows, int64_t cols, int64_t ld,
                                const int64_t* __restrict__ ptr, int32_t* __restrict__ col, float* __restrict__ val) {
    const int64_t r = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (r >= rows) return;
    int64_t pos = ptr[r];
    for (int64_t j0 = 0; j0 < cols; j0 += 32) {
        const int64_t j = j0 + lane;
        const float v = j < cols ? X[r * ld + j] : 0.f;
        const unsigned m = __ballot_sync(0xffffffffu, v != 0.f);
        if (v != 0.f) {
            const int64_t k = pos + __popc(m & ((1u << lane) - 1u));
            col[k] = (int32_t)j; val[k] = v;
        }
        pos += __popc(m);
    }
}

// Yt[k][q] = hi[q][k] + lo[q][k] (q < nq, else 0): the plan operand, element-major, so the SpMM lanes (= plans) read it coalesced
__global__ void transpose_sum_kernel(const float* __restrict__ hi, const float* __restrict__ lo, int nq, int64_t K, int64_t ld,
                                     float* __restrict__ Yt, int ldq) {
    __shared__ float t[32][33];
    const int64_t k0 = (int64_t)blockIdx.x * 32; const int q0 = blockIdx.y * 32;
    for (int y = threadIdx.y; y < 32; y += 8) {
        const int q = q0 + y; const int64_t k = k0 + threadIdx.x;
        t[y][threadIdx.x] = (q < nq && k < K) ? hi[(int64_t)q * ld + k] + lo[(int64_t)q * ld + k] : 0.f;
    }
    __syncthreads();
    for (int y = threadIdx.y; y < 32; y += 8) {
        const int64_t k = k0 + y; const int q = q0 + threadIdx.x;
        if (k < K && q < ldq) Yt[k * ldq + q] = t[threadIdx.x][y];
    }
}

// out = X . Y^T for CSR X [M][K] and Yt [K][ldq] (ldq = 32 * qc plans).  Block = 32 rows, 4 warps; a warp owns rows
// w, w+4, ..; lanes = plans.  The non-zeros of a row are read 32 at a time (coalesced) and broadcast by shuffles.
// Results go through shared memory so the stores are coalesced along the rows.
//   K1_LAYOUT = false: out[q * out_ld + m]                                  (Q buffer [plan][point])
//   K1_LAYOUT = true : out[(((m / 128) * splits + blockIdx.y) * n_mma + q) * 128 + m % 128]   (the partial-sum layout K2a reads;
//                      the rows of Phi^T are long, N * density non-zeros, so each is cut into `splits` segments = slots)
template <bool K1_LAYOUT>
__global__ void __launch_bounds__(128) csr_spmm_kernel(const int64_t* __restrict__ ptr, const int32_t* __restrict__ col,
                                                       const float* __restrict__ val, int64_t M, const float* __restrict__ Yt,
                                                       int ldq, int nq, float* __restrict__ out, int64_t out_ld, int n_mma, int splits) {
    extern __shared__ float tile[];                       // [ldq][33]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int qc = ldq >> 5;                              // <= 8
    const int64_t m0 = (int64_t)blockIdx.x * 32;
    for (int rr = warp; rr < 32; rr += 4) {
        const int64_t m = m0 + rr;
        float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (m < M) {
            const int64_t r0 = ptr[m], len = ptr[m + 1] - r0;
            const int64_t kb = r0 + len * blockIdx.y / splits, ke = r0 + len * (blockIdx.y + 1) / splits;
            for (int64_t k0 = kb; k0 < ke; k0 += 32) {
                const int cnt = (int)min((int64_t)32, ke - k0);
                const int myc = lane < cnt ? col[k0 + lane] : 0;
                const float myv = lane < cnt ? val[k0 + lane] : 0.f;
                for (int t = 0; t < cnt; ++t) {
                    const int c = __shfl_sync(0xffffffffu, myc, t);
                    const float v = __shfl_sync(0xffffffffu, myv, t);
                    const float* y = Yt + (int64_t)c * ldq + lane;
#pragma unroll
                    for (int cc = 0; cc < 8; ++cc)
                        if (cc < qc) acc[cc] = fmaf(v, y[cc * 32], acc[cc]);
                }
            }
        }
#pragma unroll
        for (int cc = 0; cc < 8; ++cc)
            if (cc < qc) tile[(cc * 32 + lane) * 33 + rr] = acc[cc];
    }
    __syncthreads();
    const int64_t m = m0 + lane;
    for (int q = warp; q < nq; q += 4) {
        if (m >= M) continue;
        const float v = tile[q * 33 + lane];
        if (K1_LAYOUT) out[(((m / kTileM) * splits + blockIdx.y) * n_mma + q) * kTileM + (m % kTileM)] = v;
        else out[(int64_t)q * out_ld + m] = v;
    }
}

admm_status build_one(admm_handle* h, const float* X, int64_t rows, int64_t cols, int64_t ld, int64_t** ptr_out,
                      int32_t** col_out, float** val_out, int64_t* nnz_out) {
    cudaStream_t st = h->stream;
    int64_t *cnt = nullptr, *ptr = nullptr; void* tmp = nullptr; size_t tmp_bytes = 0;
    if (cudaMalloc(&cnt, (size_t)(rows + 1) * 8) != cudaSuccess || cudaMalloc(&ptr, (size_t)(rows + 1) * 8) != cudaSuccess) {
        if (cnt) cudaFree(cnt);
        h->err = "CSR row pointer allocation failed"; return ADMM_ENOMEM;
    }
    cudaMemsetAsync(cnt, 0, (size_t)(rows + 1) * 8, st);
    row_count_kernel<<<(unsigned)cdiv(rows, 8), 256, 0, st>>>(X, rows, cols, ld, cnt);
    cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, cnt, ptr, (int)(rows + 1), st);
    if (cudaMalloc(&tmp, tmp_bytes) != cudaSuccess) { cudaFree(cnt); cudaFree(ptr); h->err = "CSR scan workspace allocation failed"; return ADMM_ENOMEM; }
    cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, cnt, ptr, (int)(rows + 1), st);
    int64_t nnz = 0;
    cudaMemcpyAsync(&nnz, ptr + rows, 8, cudaMemcpyDeviceToHost, st);
    cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(tmp); cudaFree(cnt);
    if (e != cudaSuccess) { cudaFree(ptr); h->err = std::string("CSR count/scan: ") + cudaGetErrorString(e); return ADMM_ECUDA; }
    int32_t* col = nullptr; float* val = nullptr;
    if (cudaMalloc(&col, (size_t)std::max<int64_t>(nnz, 1) * 4) != cudaSuccess || cudaMalloc(&val, (size_t)std::max<int64_t>(nnz, 1) * 4) != cudaSuccess) {
        if (col) cudaFree(col);
        cudaFree(ptr); h->err = "CSR value allocation failed"; return ADMM_ENOMEM;
    }
    row_fill_kernel<<<(unsigned)cdiv(rows, 8), 256, 0, st>>>(X, rows, cols, ld, ptr, col, val);
    *ptr_out = ptr; *col_out = col; *val_out = val; *nnz_out = nnz;
    return ADMM_OK;
}

}  // namespace

// zero the entries below csr_rel_threshold * max|Phi| in the row-major setup copy (before S is formed)
admm_status csr_threshold(admm_handle* h) {
    cudaStream_t st = h->stream;
    unsigned int* d_max = nullptr; unsigned int hmax = 0;
    if (cudaMalloc(&d_max, 4) != cudaSuccess) { h->err = "allocation failed"; return ADMM_ENOMEM; }
    cudaMemsetAsync(d_max, 0, 4, st);
    const int64_t count = h->N * h->ldn;
    absmax_kernel<<<1024, 256, 0, st>>>(h->d_phi, count, d_max);
    cudaMemcpyAsync(&hmax, d_max, 4, cudaMemcpyDeviceToHost, st);
    cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(d_max);
    if (e != cudaSuccess) { h->err = std::string("CSR threshold: ") + cudaGetErrorString(e); return ADMM_ECUDA; }
    float mx; memcpy(&mx, &hmax, 4);
    h->csr_tau = h->opt.csr_rel_threshold * mx;
    threshold_kernel<<<(unsigned)cdiv(count, 256), 256, 0, st>>>(h->d_phi, count, h->csr_tau);
    return ADMM_OK;
}

// CSR of Phi (from d_phi) and of Phi^T (from d_phiT); the dense copies are the caller's to free afterwards
admm_status csr_build(admm_handle* h) {
    admm_status s = build_one(h, h->d_phi, h->N, h->n, h->ldn, &h->d_csr_ptr, &h->d_csr_col, &h->d_csr_val, &h->csr_nnz);
    if (s != ADMM_OK) return s;
    int64_t nnzT = 0;
    s = build_one(h, h->d_phiT, h->n, h->N, h->ldN, &h->d_csrT_ptr, &h->d_csrT_col, &h->d_csrT_val, &nnzT);
    if (s != ADMM_OK) return s;
    if (nnzT != h->csr_nnz) { h->err = "CSR: nnz(Phi) != nnz(Phi^T)"; return ADMM_ECUDA; }
    return ADMM_OK;
}

// W partials = Phi^T . G for the slots [slot0, slot0 + nact)  (layout of K1's partial sums with one slot per m-tile)
void launch_csr_k1(admm_handle* h, int slot0, int nact, int n_mma, cudaStream_t s) {
    const int ldq = (int)cdiv(nact, 32) * 32;
    const float* hi = reinterpret_cast<const float*>(h->d_ghi) + (int64_t)slot0 * h->ldN;
    const float* lo = reinterpret_cast<const float*>(h->d_glo) + (int64_t)slot0 * h->ldN;
    transpose_sum_kernel<<<dim3((unsigned)cdiv(h->N, 32), (unsigned)(ldq / 32)), dim3(32, 8), 0, s>>>(hi, lo, nact, h->N, h->ldN, h->d_small_t, ldq);
    const int splits = h->grid_k1;          // partial-sum slots per m-tile (api.cu)
    csr_spmm_kernel<true><<<dim3((unsigned)cdiv(h->n, 32), (unsigned)splits), 128, (size_t)ldq * 33 * 4, s>>>(
        h->d_csrT_ptr, h->d_csrT_col, h->d_csrT_val, h->n, h->d_small_t, ldq, nact, h->d_partial, 0, n_mma, splits);
    h->launch_count += 2;
}
// qbuf[plan][point] = Phi . V for the nact plans whose operand starts at vhi / vlo
void launch_csr_k3(admm_handle* h, int nact, const float* vhi, const float* vlo, float* qbuf, cudaStream_t s) {
    const int ldq = (int)cdiv(nact, 32) * 32;
    transpose_sum_kernel<<<dim3((unsigned)cdiv(h->n, 32), (unsigned)(ldq / 32)), dim3(32, 8), 0, s>>>(vhi, vlo, nact, h->n, h->ldn, h->d_small_t, ldq);
    csr_spmm_kernel<false><<<(unsigned)cdiv(h->N, 32), 128, (size_t)ldq * 33 * 4, s>>>(h->d_csr_ptr, h->d_csr_col, h->d_csr_val, h->N,
                                                                                       h->d_small_t, ldq, nact, qbuf, h->ldN, 0, 1);
    h->launch_count += 2;
}
