// adamw_math.cuh -- the per-coordinate AdamW update of Algorithm 1 lines 7-10 and the
// storage conversions of line 11, in fp32.  The fused epilogue and the unfused test kernel
// (forge_adamw_from_g) inline exactly these functions; every operation is an explicit
// round-to-nearest instruction so the compiler cannot contract or reassociate them differently in
// the two kernels -- that is what makes "store-G + this" bit-identical to the fused path
// (PAPER.md:294).
//
// Everything works on PAIRS of coordinates held in one 64-bit register: sm_100 has packed fp32
// instructions (add/mul/fma.rn.f32x2 -> FADD2/FMUL2/FFMA2) that issue once for two IEEE-identical
// results, halving the issue slots and register-bandwidth of the epilogue arithmetic.
#pragma once
#include <cstdint>
#include <cuda_bf16.h>

namespace forge {

// Scalars precomputed on the host in double, then rounded to float once.
struct AdamWScalars {
    float beta1, one_minus_beta1;   // 1-beta exact in fp32 (Sterbenz)
    float beta2, one_minus_beta2;
    // W' = (1 - lr wd) W - step m' / (sqrt(v') c + eps), step = lr/(1-beta1^t), c = 1/sqrt(1-beta2^t), is evaluated as
    // decay W + m' * rcp(nd_c sqrt(v') + nd_eps) with the step size folded into the (negated) denominator: one multiply
    // less per element and one rounding less.  lr = 0 (or a step size too small for fp32): nd_c = 0, nd_eps = -inf,
    // the reciprocal is -0 and W' = decay W.
    float nd_c;                     // -(1/sqrt(1-beta2^t)) / step
    float nd_eps;                   // -eps / step
    float decay;                    // 1 - lr*wd   (decoupled decay on the pre-update W)
    // int8 moments work on the SCALED moments m'' = m'/(1-beta1), v'' = v'/(1-beta2) (adamw_moments2_qs): one FMA
    // each instead of a multiply and an FMA; the codes are scale-invariant and the factors fold into constants
    float q_b1, q_b2;               // beta/(1-beta)
    float nq_c;                     // -sqrt(1-beta2) / (sqrt(1-beta2^t) (1-beta1) step):  m'/(sqrt(v'/bc2)+eps) = m''/(sqrt(v'') q_c + q_eps)
    float nq_eps;                   // -eps / ((1-beta1) step)
};

// ------------------------------------------------------------------ packed fp32 pairs ------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f32x2 pk2u(uint32_t lo, uint32_t hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
    return r;
}
__device__ __forceinline__ f32x2 bc2(float x) { return pk2(x, x); }
__device__ __forceinline__ float lo2(f32x2 p) {
    float a;
    asm("mov.b64 {%0, _}, %1;" : "=f"(a) : "l"(p));
    return a;
}
__device__ __forceinline__ float hi2(f32x2 p) {
    float b;
    asm("mov.b64 {_, %0}, %1;" : "=f"(b) : "l"(p));
    return b;
}
__device__ __forceinline__ uint32_t lo2u(f32x2 p) { return __float_as_uint(lo2(p)); }
__device__ __forceinline__ uint32_t hi2u(f32x2 p) { return __float_as_uint(hi2(p)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// The square root and the reciprocal are the hardware approximations (MUFU.SQRT / MUFU.RCP,
// <= 1-2 ulp of fp32 each): the ratio is off by <= ~2^-21 relative, i.e. W' by <= lr*2^-21*|ratio|,
// four orders of magnitude below a bf16 ulp of W; the IEEE sequences cost ~4x the instructions.
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

// m' = b1 m + (1-b1) g ; v' = b2 v + (1-b2) g^2                       (Alg. 1 lines 7-8)
__device__ __forceinline__ void adamw_moments2(const AdamWScalars &h, f32x2 g, f32x2 &m, f32x2 &v) {
    m = fma2(bc2(h.beta1), m, mul2(bc2(h.one_minus_beta1), g));
    v = fma2(bc2(h.beta2), v, mul2(mul2(bc2(h.one_minus_beta2), g), g));
}
// the same with int8 state: the stored moment is code * (a/L); beta * (a/L) is one per-block constant
// (bm = fp32(beta1 * fp32(a_m/127)), bv likewise), so dequantisation costs no extra instruction
__device__ __forceinline__ void adamw_moments2_q(const AdamWScalars &h, f32x2 g, f32x2 code_m, f32x2 code_v,
                                                 float bm, float bv, f32x2 &m, f32x2 &v) {
    m = fma2(bc2(bm), code_m, mul2(bc2(h.one_minus_beta1), g));
    v = fma2(bc2(bv), code_v, mul2(mul2(bc2(h.one_minus_beta2), g), g));
}
// int8 state on the scaled moments: m'' = m'/(1-b1) = (b1/(1-b1) a/L) code + g, v'' = (b2/(1-b2) a/L) code + g^2.
// bmq = fp32(q_b1 * fp32(a_m/127)), bvq likewise.  max|m''| (1-b1) is the stored block absmax; code = rint(m'' L/max|m''|).
__device__ __forceinline__ void adamw_moments2_qs(f32x2 g, f32x2 code_m, f32x2 code_v, float bmq, float bvq, f32x2 &m, f32x2 &v) {
    m = fma2(bc2(bmq), code_m, g);
    v = fma2(bc2(bvq), code_v, mul2(g, g));
}
__device__ __forceinline__ void adamw_weight2_s(const AdamWScalars &h, f32x2 m, f32x2 v, f32x2 &w) {
    const f32x2 sq = pk2(sqrt_fast(lo2(v)), sqrt_fast(hi2(v)));
    const f32x2 nden = fma2(sq, bc2(h.nq_c), bc2(h.nq_eps));
    w = fma2(m, pk2(rcp_fast(lo2(nden)), rcp_fast(hi2(nden))), mul2(bc2(h.decay), w));
}
// W' = (1 - lr wd) W - lr * (m'/bc1) / (sqrt(v'/bc2) + eps)          (Alg. 1 lines 9-10)
// sqrt(v'/bc2) is evaluated as sqrt(v') * (1/sqrt(bc2)); the step size lr/bc1 is folded into the denominator (see
// AdamWScalars); W' uses the unrounded m', v'.
__device__ __forceinline__ void adamw_weight2(const AdamWScalars &h, f32x2 m, f32x2 v, f32x2 &w) {
    const f32x2 sq = pk2(sqrt_fast(lo2(v)), sqrt_fast(hi2(v)));
    const f32x2 nden = fma2(sq, bc2(h.nd_c), bc2(h.nd_eps));
    w = fma2(m, pk2(rcp_fast(lo2(nden)), rcp_fast(hi2(nden))), mul2(bc2(h.decay), w));
}
__device__ __forceinline__ void adamw_update2(const AdamWScalars &h, f32x2 g, f32x2 &w, f32x2 &m, f32x2 &v) {
    adamw_moments2(h, g, m, v);
    adamw_weight2(h, m, v, w);
}

// ------------------------------------------------------------------ bf16 packing -----------
__device__ __forceinline__ float bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }
__device__ __forceinline__ f32x2 bf16x2_to_f32x2(uint32_t u) { return pk2u(u << 16, u & 0xFFFF0000u); }
// two floats -> packed bf16x2 (round to nearest even), `lo` in the low half
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&t);
}
__device__ __forceinline__ uint32_t f32x2_to_bf16x2(f32x2 p) { return pack_bf16(lo2(p), hi2(p)); }

// ------------------------------------------------------------------ stochastic-rounding store
// The paper's "SR-store" recipe: the bf16 weight is committed by stochastic rounding.
// 16 random bits per element from a counter-based generator keyed (seed, step, stream, row, col) through the
// murmur3 finaliser (reading S16); out = (bits(x) + r16) >> 16 rounds the fp32 value away from zero with
// probability (low 16 bits) / 65536.  Inf / NaN take the RNE path.
__device__ __forceinline__ uint32_t fmix32(uint32_t h) {
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    return h;
}
__host__ __device__ inline uint32_t sr_inner_key_host(uint32_t seed_hi, uint32_t step, uint32_t stream) {
    uint32_t h = seed_hi ^ (step * 0x85EBCA77u) ^ (stream * 0xC2B2AE3Du);
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    return h;
}
__device__ __forceinline__ uint32_t sr_row_key(uint32_t row, uint32_t seed_lo, uint32_t inner) {
    return fmix32((row * 0x9E3779B1u) ^ seed_lo ^ inner);
}
__device__ __forceinline__ uint32_t sr_bf16(float x, uint32_t rowkey, uint32_t col) {
    const uint32_t b = __float_as_uint(x);
    if ((b & 0x7F800000u) == 0x7F800000u) return pack_bf16(x, 0.0f) & 0xFFFFu;
    return (b + (fmix32(rowkey ^ (col * 0x27D4EB2Fu)) >> 16)) >> 16;
}
__device__ __forceinline__ uint32_t f32x2_to_bf16x2_sr(f32x2 p, uint32_t rowkey, uint32_t col) {
    return sr_bf16(lo2(p), rowkey, col) | (sr_bf16(hi2(p), rowkey, col + 1u) << 16);
}

// ------------------------------------------------------------------ fp8 (e4m3) moments ------
// PAPER.md:359-362 "fp8 states (per-tensor scale) ... delayed scaling" (reading S17): stored code =
// e4m3(x / s) with one fp32 scale per tensor; the hardware converters do the work.
// two e4m3 codes (low 16 bits of `pair`) -> two floats holding the code values
__device__ __forceinline__ f32x2 e4m3x2_to_f32x2(uint32_t pair) {
    uint32_t h2;
    asm("{\n\t.reg .b16 t;\n\tcvt.u16.u32 t, %1;\n\tcvt.rn.f16x2.e4m3x2 %0, t;\n\t}\n" : "=r"(h2) : "r"(pair));
    float lo, hi;
    asm("{\n\t.reg .b16 a, b;\n\tmov.b32 {a, b}, %2;\n\tcvt.f32.f16 %0, a;\n\tcvt.f32.f16 %1, b;\n\t}\n"
        : "=f"(lo), "=f"(hi)
        : "r"(h2));
    return pk2(lo, hi);
}
// two floats -> two e4m3 codes (round to nearest even, saturate to +-448), `lo` in the low byte
__device__ __forceinline__ uint32_t f32x2_to_e4m3x2(f32x2 p) {
    uint32_t r;
    asm("{\n\t.reg .b16 t;\n\tcvt.rn.satfinite.e4m3x2.f32 t, %2, %1;\n\tcvt.u32.u16 %0, t;\n\t}\n"
        : "=r"(r)
        : "f"(lo2(p)), "f"(hi2(p)));
    return r;
}
__device__ __forceinline__ float fp8_inv_scale(float s) { return s > 0.0f ? __fdiv_rn(1.0f, s) : 0.0f; }

// ------------------------------------------------------------------ int8 blockwise ---------
// PAPER.md:316 with BASELINE.json's 256-blocks: scale a = block absmax (fp32);
// m code = rint(x * (127/a)) in [-127,127]; v code = max(1, rint(x * (255/a))) in [1,255];
// a == 0 -> all codes 0.  The quotient L/a is rounded to fp32; the code is the round-to-nearest-even
// integer of the EXACT product x * fp32(L/a).
//
// No integer<->float conversion instruction is used (they run at a quarter of the FMA rate):
//   code -> float : the byte is spliced under the exponent of 2^23 (one PRMT), then 2^23 (+128 for
//                   the sign-flipped m code) is subtracted -- exact;
//   float -> code : fma(x, inv, 1.5*2^23) rounds the exact product to an integer (ulp = 1, ties to
//                   even) whose two's-complement low byte sits in the low byte of the result.
// |x * inv| <= L(1 + 2^-23) rounds to at most L, so no clamp is needed for finite state.
constexpr float kMagicSplice = 8388608.0f;        // 2^23  = 0x4B000000
constexpr float kMagicRound = 12582912.0f;        // 1.5 * 2^23
__device__ __forceinline__ float quant_inv_scale(float absmax, float levels) {
    return absmax > 0.0f ? __fdiv_rn(levels, absmax) : 0.0f;
}
__device__ __forceinline__ float dequant_step(float absmax, float levels) {
    return __fdiv_rn(absmax, levels);
}
// four packed codes -> four floats holding the integer code values
__device__ __forceinline__ void codes4_to_f32(uint32_t word, bool is_signed, f32x2 &c01, f32x2 &c23) {
    const uint32_t u = is_signed ? (word ^ 0x80808080u) : word;
    const float bias = is_signed ? -(kMagicSplice + 128.0f) : -kMagicSplice;
    c01 = add2(pk2u(__byte_perm(u, 0x4B000000u, 0x7540), __byte_perm(u, 0x4B000000u, 0x7541)), bc2(bias));
    c23 = add2(pk2u(__byte_perm(u, 0x4B000000u, 0x7542), __byte_perm(u, 0x4B000000u, 0x7543)), bc2(bias));
}
// pair of values -> pair of floats whose low bytes are the codes
__device__ __forceinline__ f32x2 quant_m2(f32x2 x, float inv) { return fma2(x, bc2(inv), bc2(kMagicRound)); }
__device__ __forceinline__ f32x2 quant_v2(f32x2 x, float inv, float floor_code /* kMagicRound + (inv > 0) */) {
    const f32x2 y = fma2(x, bc2(inv), bc2(kMagicRound));
    return pk2(fmaxf(lo2(y), floor_code), fmaxf(hi2(y), floor_code));
}
__device__ __forceinline__ float quant_v_floor(float inv) { return inv > 0.0f ? kMagicRound + 1.0f : kMagicRound; }
__device__ __forceinline__ uint32_t pack_codes4(f32x2 q01, f32x2 q23) {
    const uint32_t t0 = __byte_perm(lo2u(q01), hi2u(q01), 0x0040), t1 = __byte_perm(lo2u(q23), hi2u(q23), 0x0040);
    return __byte_perm(t0, t1, 0x5410);
}

}  // namespace forge
