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
    float g[8], w[8], m[8], v[8];
    float a_m_old = 0.f, a_v_old = 0.f;
    if (active) {
        const float4 g0 = *reinterpret_cast<const float4 *>(G + base), g1 = *reinterpret_cast<const float4 *>(G + base + 4);
        g[0] = g0.x; g[1] = g0.y; g[2] = g0.z; g[3] = g0.w; g[4] = g1.x; g[5] = g1.y; g[6] = g1.z; g[7] = g1.w;
        const uint4 wq = *reinterpret_cast<const uint4 *>(W + base);
        w[0] = bf16lo(wq.x); w[1] = bf16hi(wq.x); w[2] = bf16lo(wq.y); w[3] = bf16hi(wq.y);
        w[4] = bf16lo(wq.z); w[5] = bf16hi(wq.z); w[6] = bf16lo(wq.w); w[7] = bf16hi(wq.w);
        if constexpr (MDT == MDT_FP32) {
            const float *mf = static_cast<const float *>(mp), *vf = static_cast<const float *>(vp);
            const float4 a = *reinterpret_cast<const float4 *>(mf + base), b = *reinterpret_cast<const float4 *>(mf + base + 4);
            const float4 c = *reinterpret_cast<const float4 *>(vf + base), d = *reinterpret_cast<const float4 *>(vf + base + 4);
            m[0] = a.x; m[1] = a.y; m[2] = a.z; m[3] = a.w; m[4] = b.x; m[5] = b.y; m[6] = b.z; m[7] = b.w;
            v[0] = c.x; v[1] = c.y; v[2] = c.z; v[3] = c.w; v[4] = d.x; v[5] = d.y; v[6] = d.z; v[7] = d.w;
        } else if constexpr (MDT == MDT_BF16) {
            const uint4 a = *reinterpret_cast<const uint4 *>(static_cast<const uint16_t *>(mp) + base);
            const uint4 c = *reinterpret_cast<const uint4 *>(static_cast<const uint16_t *>(vp) + base);
            m[0] = bf16lo(a.x); m[1] = bf16hi(a.x); m[2] = bf16lo(a.y); m[3] = bf16hi(a.y);
            m[4] = bf16lo(a.z); m[5] = bf16hi(a.z); m[6] = bf16lo(a.w); m[7] = bf16hi(a.w);
            v[0] = bf16lo(c.x); v[1] = bf16hi(c.x); v[2] = bf16lo(c.y); v[3] = bf16hi(c.y);
            v[4] = bf16lo(c.z); v[5] = bf16hi(c.z); v[6] = bf16lo(c.w); v[7] = bf16hi(c.w);
        } else {
            a_m_old = m_scale[base / 256];
            a_v_old = v_scale[base / 256];
            const float dm = dequant_step(a_m_old, 127.0f), dv = dequant_step(a_v_old, 255.0f);
            const uint2 a = *reinterpret_cast<const uint2 *>(static_cast<const uint8_t *>(mp) + base);
            const uint2 c = *reinterpret_cast<const uint2 *>(static_cast<const uint8_t *>(vp) + base);
            const uint32_t aw[2] = {a.x, a.y}, cw[2] = {c.x, c.y};
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int mc = static_cast<int>(static_cast<int8_t>((aw[e >> 2] >> (8 * (e & 3))) & 0xFFu));
                const int vc = static_cast<int>((cw[e >> 2] >> (8 * (e & 3))) & 0xFFu);
                m[e] = __fmul_rn(static_cast<float>(mc), dm);
                v[e] = __fmul_rn(static_cast<float>(vc), dv);
            }
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) adamw_update(hp, g[e], w[e], m[e], v[e]);
        *reinterpret_cast<uint4 *>(W + base) = make_uint4(pack_bf16(w[0], w[1]), pack_bf16(w[2], w[3]),
                                                          pack_bf16(w[4], w[5]), pack_bf16(w[6], w[7]));
        if constexpr (MDT == MDT_FP32) {
            float *mf = static_cast<float *>(mp), *vf = static_cast<float *>(vp);
            *reinterpret_cast<float4 *>(mf + base) = make_float4(m[0], m[1], m[2], m[3]);
            *reinterpret_cast<float4 *>(mf + base + 4) = make_float4(m[4], m[5], m[6], m[7]);
            *reinterpret_cast<float4 *>(vf + base) = make_float4(v[0], v[1], v[2], v[3]);
            *reinterpret_cast<float4 *>(vf + base + 4) = make_float4(v[4], v[5], v[6], v[7]);
        } else if constexpr (MDT == MDT_BF16) {
            *reinterpret_cast<uint4 *>(static_cast<uint16_t *>(mp) + base) =
                make_uint4(pack_bf16(m[0], m[1]), pack_bf16(m[2], m[3]), pack_bf16(m[4], m[5]), pack_bf16(m[6], m[7]));
            *reinterpret_cast<uint4 *>(static_cast<uint16_t *>(vp) + base) =
                make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]), pack_bf16(v[6], v[7]));
        }
    }
    if constexpr (MDT == MDT_INT8) {
        // n_elems % 256 == 0, so a warp is either fully active or fully idle
        float pm = 0.f, pv = 0.f;
        if (active) {
#pragma unroll
            for (int e = 0; e < 8; ++e) { pm = fmaxf(pm, fabsf(m[e])); pv = fmaxf(pv, fabsf(v[e])); }
        }
        const float a_m = warp_max(pm), a_v = warp_max(pv);
        if (active) {
            const float inv_m = quant_inv_scale(a_m, 127.0f), inv_v = quant_inv_scale(a_v, 255.0f);
            uint32_t mo[2] = {0, 0}, vo[2] = {0, 0};
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                mo[e >> 2] |= (static_cast<uint32_t>(quant_m_code(m[e], inv_m)) & 0xFFu) << (8 * (e & 3));
                vo[e >> 2] |= (static_cast<uint32_t>(quant_v_code(v[e], inv_v)) & 0xFFu) << (8 * (e & 3));
            }
            *reinterpret_cast<uint2 *>(static_cast<uint8_t *>(mp) + base) = make_uint2(mo[0], mo[1]);
            *reinterpret_cast<uint2 *>(static_cast<uint8_t *>(vp) + base) = make_uint2(vo[0], vo[1]);
            if ((threadIdx.x & 31) == 0) {
                m_scale[base / 256] = a_m;
                v_scale[base / 256] = a_v;
            }
        }
    }
}

}  // namespace forge
