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
#include "tc_ptx.cuh"

struct Epi1Out {
    float s_new;
    float g_hi, g_lo;
};

// one (point, plan) element of epilogue-1.  acc[0..4] += residual terms when `resid`.
__device__ __forceinline__ Epi1Out epi1_element(float s_old, float q, float a, float cr, float ub, bool resid, float* acc) {
    float z_old = fminf(fmaxf(s_old, 0.0f), ub);
    float s_new = z_old - cr - a * q;
    float z_new = fminf(fmaxf(s_new, 0.0f), ub);
    float g = a * (2.0f * z_new - s_new - cr);
    Epi1Out o;
    o.s_new = s_new;
    o.g_hi = tc::tf32_rna(g);
    o.g_lo = tc::tf32_rna(g - o.g_hi);      // rounded here: the tensor core would otherwise cut lo's low bits toward zero
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
