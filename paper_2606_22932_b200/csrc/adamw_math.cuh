// adamw_math.cuh -- the per-coordinate AdamW update of Algorithm 1 lines 7-10 and the
// storage conversions of line 11, in fp32.  The fused epilogue and the unfused test kernel
// (forge_adamw_from_g) inline exactly these functions; every operation is an explicit
// round-to-nearest intrinsic so the compiler cannot contract or reassociate them differently in
// the two kernels -- that is what makes "store-G + this" bit-identical to the fused path
// (PAPER.md:294).
#pragma once
#include <cstdint>
#include <cuda_bf16.h>

namespace forge {

// Scalars precomputed on the host in double, then rounded to float once.
struct AdamWScalars {
    float beta1, one_minus_beta1;   // 1-beta exact in fp32 (Sterbenz)
    float beta2, one_minus_beta2;
    float step_size;                // lr / (1 - beta1^t)
    float inv_sqrt_bc2;             // 1 / sqrt(1 - beta2^t)
    float eps;
    float decay;                    // 1 - lr*wd   (decoupled decay on the pre-update W)
};

// m' = b1 m + (1-b1) g ; v' = b2 v + (1-b2) g^2 ;
// W' = (1 - lr wd) W - lr * (m'/bc1) / (sqrt(v'/bc2) + eps)          (Alg. 1 lines 7-10)
// sqrt(v'/bc2) is evaluated as sqrt(v') * (1/sqrt(bc2)); W' uses the unrounded m', v'.
// The square root and the reciprocal are the hardware approximations (MUFU.SQRT / MUFU.RCP,
// <= 1-2 ulp of fp32 each): the ratio is off by <= ~2^-21 relative, i.e. W' by <= lr*2^-21*|ratio|,
// four orders of magnitude below a bf16 ulp of W; the IEEE sequences cost ~4x the instructions
// and made the epilogue, not HBM, the bottleneck (profiles/r01_fp32_first.md).
__device__ __forceinline__ float sqrt_fast(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_fast(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ void adamw_update(const AdamWScalars &h, float g, float &w, float &m,
                                             float &v) {
    m = __fmaf_rn(h.beta1, m, __fmul_rn(h.one_minus_beta1, g));
    v = __fmaf_rn(h.beta2, v, __fmul_rn(__fmul_rn(h.one_minus_beta2, g), g));
    const float denom = __fmaf_rn(sqrt_fast(v), h.inv_sqrt_bc2, h.eps);
    const float ratio = __fmul_rn(m, rcp_fast(denom));
    w = __fmaf_rn(-h.step_size, ratio, __fmul_rn(h.decay, w));
}

// ------------------------------------------------------------------ bf16 packing -----------
__device__ __forceinline__ float bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }
// two floats -> packed bf16x2 (round to nearest even), `lo` in the low half
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&t);
}

// ------------------------------------------------------------------ int8 blockwise ---------
// PAPER.md:316 with BASELINE.json's 256-blocks: scale a = block absmax (fp32);
// m code = rint(x * (127/a)) in [-127,127]; v code = max(1, rint(x * (255/a))) in [1,255];
// a == 0 -> all codes 0.  Quotient and product each rounded to fp32, ties to even.
__device__ __forceinline__ float quant_inv_scale(float absmax, float levels) {
    return absmax > 0.0f ? __fdiv_rn(levels, absmax) : 0.0f;
}
__device__ __forceinline__ int quant_m_code(float x, float inv) {
    int c = __float2int_rn(__fmul_rn(x, inv));
    return max(-127, min(127, c));
}
__device__ __forceinline__ int quant_v_code(float x, float inv) {
    int c = __float2int_rn(__fmul_rn(x, inv));
    c = max(1, min(255, c));
    return inv > 0.0f ? c : 0;
}
__device__ __forceinline__ float dequant_step(float absmax, float levels) {
    return __fdiv_rn(absmax, levels);
}

}  // namespace forge
