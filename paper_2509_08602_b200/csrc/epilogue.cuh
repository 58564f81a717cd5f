// Element-wise pieces of the ADMM iteration in single-state form.
//
// The stored state of block 1 is s1 = x1 + y1 (previous y).  From (4b)/(4c), PAPER.md:73-76:
//     z1 = clip(s1, 0, u)            y1 = s1 - z1
// and (7), gives the next state
//     s1+ = x1+ + y1 = z1 - c/rho - A^T v
// with A^T v = a_i * Q[i], Q = Phi (R o v), a_i = sigma_i D_i (class sign / threshold / count folded).
// The operand of the next A r1 product is r1 = z1+ - y1+ - c/rho = 2 z1+ - s1+ - c/rho, scaled by a_i.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include "tc_ptx.cuh"

// A small-operand element x as a hi/lo pair for the tensor cores: fp32 containers on the tf32 grid (hi = rna(x),
// lo = rna(x - hi): 21 bits kept, both rounded here so the hardware's operand truncation never bites), or a bf16
// pair (16 bits kept) for ADMM_STORAGE_BF16.
__device__ __forceinline__ void emit_small(void* hi, void* lo, int64_t rowbase, int64_t col, float x, bool bf16) {
    const int64_t idx = (bf16 ? 2 * rowbase : rowbase) + col;      // same row pitch in bytes for both element types
    if (bf16) {
        const __nv_bfloat16 h = __float2bfloat16_rn(x);
        reinterpret_cast<__nv_bfloat16*>(hi)[idx] = h;
        reinterpret_cast<__nv_bfloat16*>(lo)[idx] = __float2bfloat16_rn(x - __bfloat162float(h));
    } else {
        const float h = tc::tf32_rna(x);
        reinterpret_cast<float*>(hi)[idx] = h;
        reinterpret_cast<float*>(lo)[idx] = tc::tf32_rna(x - h);
    }
}
__device__ __forceinline__ void emit_small(void* hi, void* lo, int64_t rowbase, int64_t col, double x, bool bf16) {
    const int64_t idx = (bf16 ? 2 * rowbase : rowbase) + col;
    if (bf16) {
        const __nv_bfloat16 h = __float2bfloat16_rn((float)x);
        reinterpret_cast<__nv_bfloat16*>(hi)[idx] = h;
        reinterpret_cast<__nv_bfloat16*>(lo)[idx] = __float2bfloat16_rn((float)(x - (double)__bfloat162float(h)));
    } else {
        const float h = tc::tf32_rn((float)x);
        reinterpret_cast<float*>(hi)[idx] = h;
        reinterpret_cast<float*>(lo)[idx] = tc::tf32_rn((float)(x - (double)h));
    }
}

struct Epi1Out {
    float s_new;
    float g;          // operand of the next A r1 product, before the hi/lo split (emit_small)
};

// one (point, plan) element of epilogue-1.  acc[0..4] += residual terms when `resid`.
__device__ __forceinline__ Epi1Out epi1_element(float s_old, float q, float a, float cr, float ub, bool resid, float* acc) {
    float z_old = fminf(fmaxf(s_old, 0.0f), ub);
    float s_new = z_old - cr - a * q;
    float z_new = fminf(fmaxf(s_new, 0.0f), ub);
    float g = a * (2.0f * z_new - s_new - cr);
    Epi1Out o;
    o.s_new = s_new;
    o.g = g;
    if (resid) {
        float y_old = s_old - z_old;
        float y_new = s_new - z_new;
        float x = s_new - y_old;
        float dp = x - z_new, dd = z_new - z_old;
        acc[0] += dp * dp;
        acc[1] += dd * dd;
        acc[2] += x * x;
        acc[3] += z_new * z_new;
        acc[4] += y_new * y_new;
    }
    return o;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
