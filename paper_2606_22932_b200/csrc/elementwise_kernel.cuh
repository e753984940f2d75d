// elementwise_kernel.cuh -- TEST/BENCH-ONLY unfused optimizer pass over a materialised fp32 G
// (the paper's standalone "FORGE optimizer kernel").  It inlines the same
// adamw_update / quantiser functions as the fused epilogue, so forge_wgrad_store_g followed by
// this kernel is bit-identical to the fused kernel.  Never on the product path.
//
// One lane owns 8 consecutive elements of a row; a warp therefore owns 256 consecutive elements,
// which in INT8 mode is exactly one quantisation block (in % 256 == 0), whose absmax is reduced
// with warp shuffles.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "adamw_math.cuh"
#include "fused_kernel.cuh"  // MDT_* enumerators only

namespace forge {

__device__ __forceinline__ float warp_max(float x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmaxf(x, __shfl_xor_sync(0xffffffffu, x, o));
    return x;
}

template <int MDT>
__global__ void __launch_bounds__(256)
forge_adamw_from_g_kernel(const float *__restrict__ G, uint16_t *__restrict__ W, void *__restrict__ mp,
                          void *__restrict__ vp, float *__restrict__ m_scale, float *__restrict__ v_scale,
                          size_t n_elems, AdamWScalars hp) {
    const size_t group = (static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x);
    const size_t base = group * 8;
    const bool active = base < n_elems;      // n_elems % 8 == 0
    f32x2 g[4], w[4], m[4], v[4];           // 8 consecutive elements as 4 coordinate pairs
    if (active) {
        const uint4 g0 = *reinterpret_cast<const uint4 *>(G + base), g1 = *reinterpret_cast<const uint4 *>(G + base + 4);
        g[0] = pk2u(g0.x, g0.y); g[1] = pk2u(g0.z, g0.w); g[2] = pk2u(g1.x, g1.y); g[3] = pk2u(g1.z, g1.w);
        const uint4 wq = *reinterpret_cast<const uint4 *>(W + base);
        w[0] = bf16x2_to_f32x2(wq.x); w[1] = bf16x2_to_f32x2(wq.y); w[2] = bf16x2_to_f32x2(wq.z); w[3] = bf16x2_to_f32x2(wq.w);
        if constexpr (MDT == MDT_FP32) {
            const float *mf = static_cast<const float *>(mp), *vf = static_cast<const float *>(vp);
            const uint4 a = *reinterpret_cast<const uint4 *>(mf + base), b = *reinterpret_cast<const uint4 *>(mf + base + 4);
            const uint4 c = *reinterpret_cast<const uint4 *>(vf + base), d = *reinterpret_cast<const uint4 *>(vf + base + 4);
            m[0] = pk2u(a.x, a.y); m[1] = pk2u(a.z, a.w); m[2] = pk2u(b.x, b.y); m[3] = pk2u(b.z, b.w);
            v[0] = pk2u(c.x, c.y); v[1] = pk2u(c.z, c.w); v[2] = pk2u(d.x, d.y); v[3] = pk2u(d.z, d.w);
#pragma unroll
            for (int e = 0; e < 4; ++e) adamw_update2(hp, g[e], w[e], m[e], v[e]);
            float *mo = static_cast<float *>(mp), *vo = static_cast<float *>(vp);
            *reinterpret_cast<uint4 *>(mo + base) = make_uint4(lo2u(m[0]), hi2u(m[0]), lo2u(m[1]), hi2u(m[1]));
            *reinterpret_cast<uint4 *>(mo + base + 4) = make_uint4(lo2u(m[2]), hi2u(m[2]), lo2u(m[3]), hi2u(m[3]));
            *reinterpret_cast<uint4 *>(vo + base) = make_uint4(lo2u(v[0]), hi2u(v[0]), lo2u(v[1]), hi2u(v[1]));
            *reinterpret_cast<uint4 *>(vo + base + 4) = make_uint4(lo2u(v[2]), hi2u(v[2]), lo2u(v[3]), hi2u(v[3]));
        } else if constexpr (MDT == MDT_BF16) {
            const uint4 a = *reinterpret_cast<const uint4 *>(static_cast<const uint16_t *>(mp) + base);
            const uint4 c = *reinterpret_cast<const uint4 *>(static_cast<const uint16_t *>(vp) + base);
            m[0] = bf16x2_to_f32x2(a.x); m[1] = bf16x2_to_f32x2(a.y); m[2] = bf16x2_to_f32x2(a.z); m[3] = bf16x2_to_f32x2(a.w);
            v[0] = bf16x2_to_f32x2(c.x); v[1] = bf16x2_to_f32x2(c.y); v[2] = bf16x2_to_f32x2(c.z); v[3] = bf16x2_to_f32x2(c.w);
#pragma unroll
            for (int e = 0; e < 4; ++e) adamw_update2(hp, g[e], w[e], m[e], v[e]);
            *reinterpret_cast<uint4 *>(static_cast<uint16_t *>(mp) + base) =
                make_uint4(f32x2_to_bf16x2(m[0]), f32x2_to_bf16x2(m[1]), f32x2_to_bf16x2(m[2]), f32x2_to_bf16x2(m[3]));
            *reinterpret_cast<uint4 *>(static_cast<uint16_t *>(vp) + base) =
                make_uint4(f32x2_to_bf16x2(v[0]), f32x2_to_bf16x2(v[1]), f32x2_to_bf16x2(v[2]), f32x2_to_bf16x2(v[3]));
        } else {
            const float bm = __fmul_rn(hp.q_b1, dequant_step(m_scale[base / 256], 127.0f));     // scaled moments m'', v''
            const float bv = __fmul_rn(hp.q_b2, dequant_step(v_scale[base / 256], 255.0f));
            const uint2 a = *reinterpret_cast<const uint2 *>(static_cast<const uint8_t *>(mp) + base);
            const uint2 c = *reinterpret_cast<const uint2 *>(static_cast<const uint8_t *>(vp) + base);
            f32x2 cm[4], cv[4];
            codes4_to_f32(a.x, true, cm[0], cm[1]);
            codes4_to_f32(a.y, true, cm[2], cm[3]);
            codes4_to_f32(c.x, false, cv[0], cv[1]);
            codes4_to_f32(c.y, false, cv[2], cv[3]);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                adamw_moments2_qs(g[e], cm[e], cv[e], bm, bv, m[e], v[e]);
                adamw_weight2_s(hp, m[e], v[e], w[e]);
            }
        }
        *reinterpret_cast<uint4 *>(W + base) = make_uint4(f32x2_to_bf16x2(w[0]), f32x2_to_bf16x2(w[1]),
                                                          f32x2_to_bf16x2(w[2]), f32x2_to_bf16x2(w[3]));
    }
    if constexpr (MDT == MDT_INT8) {
        // n_elems % 256 == 0, so a warp is either fully active or fully idle
        float pm = 0.f, pv = 0.f;
        if (active) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                pm = fmaxf(pm, fmaxf(fabsf(lo2(m[e])), fabsf(hi2(m[e]))));
                pv = fmaxf(pv, fmaxf(lo2(v[e]), hi2(v[e])));
            }
        }
        const float a_m = warp_max(pm), a_v = warp_max(pv);
        if (active) {
            const float inv_m = quant_inv_scale(a_m, 127.0f), inv_v = quant_inv_scale(a_v, 255.0f);
            const float v_floor = quant_v_floor(inv_v);
            const uint32_t m0 = pack_codes4(quant_m2(m[0], inv_m), quant_m2(m[1], inv_m));
            const uint32_t m1 = pack_codes4(quant_m2(m[2], inv_m), quant_m2(m[3], inv_m));
            const uint32_t v0 = pack_codes4(quant_v2(v[0], inv_v, v_floor), quant_v2(v[1], inv_v, v_floor));
            const uint32_t v1 = pack_codes4(quant_v2(v[2], inv_v, v_floor), quant_v2(v[3], inv_v, v_floor));
            *reinterpret_cast<uint2 *>(static_cast<uint8_t *>(mp) + base) = make_uint2(m0, m1);
            *reinterpret_cast<uint2 *>(static_cast<uint8_t *>(vp) + base) = make_uint2(v0, v1);
            if ((threadIdx.x & 31) == 0) {          // stored absmax of m', v' = (1 - beta) max of the scaled moments
                m_scale[base / 256] = __fmul_rn(hp.one_minus_beta1, a_m);
                v_scale[base / 256] = __fmul_rn(hp.one_minus_beta2, a_v);
            }
        }
    }
}

}  // namespace forge
