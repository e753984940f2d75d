// family_math.cuh -- the other coordinate-wise ("regime 1") optimizer families of PAPER.md:267 Definition 1
// as ONE parametrised per-coordinate update: SGD, SGD with momentum / Nesterov, Lion, RMSprop, Adagrad,
// Adamax, NAdam, RAdam (App. I; the rules are torch.optim's, Lion is Chen et al. 2023).
// Every family is a choice of host-precomputed scalars (forge_api.cu::make_family) in
//
//     g' = g + cwd * w                                   coupled (L2) weight decay, 0 when decoupled / none
//     m' = a1 * m + a2 * g'                              momentum-like state, if the family has one
//     v' = b1 * v + b2 * g'^2         (V_EMA)            second-moment state, if the family has one
//     v' = max(b1 * v, |g'| + e2)     (V_MAX, Adamax)
//     n  = c1 * m' + c2 * g'          or   sign(l1 * m + l2 * g)   (Lion: interpolation of the OLD m)
//     d  = sqrt(v') * e1 + e2  (V_EMA) | v' (V_MAX) | 1 (no denominator)
//     w' = decay * w - step * n / d
//
// in fp32 on packed pairs (FFMA2 / FMUL2), W' from the unrounded new state (reading S3).
#pragma once
#include "adamw_math.cuh"

namespace forge {

enum : int { V_NONE = 0, V_EMA = 1, V_MAX = 2 };

struct FamilyScalars {
    float cwd;
    float a1, a2;
    float b1, b2;
    float c1, c2;
    float l1, l2;
    float e1, e2;
    float step, decay;
    int32_t has_m;       // state 0 is momentum-like
    int32_t v_mode;      // V_NONE / V_EMA / V_MAX; the v-like state is state 1, or state 0 when has_m == 0
    int32_t lion;        // direction is a sign
    int32_t has_denom;   // divide the direction by d
    int32_t kind;        // FK_* : the compile-time structure the epilogue dispatches on
};

__device__ __forceinline__ float sign_or_zero(float c) { return static_cast<float>((c > 0.0f) - (c < 0.0f)); }

// One coordinate pair.  The family's structure is a compile-time choice (the epilogue switches ONCE per
// sub-block on FamilyScalars::kind), so the inner loops carry no branches.  m / v are ignored (and left
// untouched) when the family does not have them.
template <bool HAS_M, int V_MODE, bool LION, bool DENOM>
__device__ __forceinline__ void family_update2(const FamilyScalars &f, f32x2 g, f32x2 &w, f32x2 &m, f32x2 &v) {
    const f32x2 gp = fma2(bc2(f.cwd), w, g);
    f32x2 n;
    if constexpr (LION) {
        const f32x2 c = fma2(bc2(f.l1), m, mul2(bc2(f.l2), g));
        n = pk2(sign_or_zero(lo2(c)), sign_or_zero(hi2(c)));
    }
    if constexpr (HAS_M) m = fma2(bc2(f.a1), m, mul2(bc2(f.a2), gp));
    if constexpr (!LION) {
        if constexpr (HAS_M) n = fma2(bc2(f.c1), m, mul2(bc2(f.c2), gp));
        else n = mul2(bc2(f.c2), gp);
    }
    if constexpr (V_MODE == V_EMA) {
        v = fma2(bc2(f.b1), v, mul2(mul2(bc2(f.b2), gp), gp));
    } else if constexpr (V_MODE == V_MAX) {
        const f32x2 dv = mul2(bc2(f.b1), v);
        v = pk2(fmaxf(lo2(dv), __fadd_rn(fabsf(lo2(gp)), f.e2)), fmaxf(hi2(dv), __fadd_rn(fabsf(hi2(gp)), f.e2)));
    }
    if constexpr (DENOM) {
        f32x2 d = v;
        if constexpr (V_MODE == V_EMA) d = fma2(pk2(sqrt_fast(lo2(v)), sqrt_fast(hi2(v))), bc2(f.e1), bc2(f.e2));
        n = mul2(n, pk2(rcp_fast(lo2(d)), rcp_fast(hi2(d))));
    }
    w = fma2(bc2(-f.step), n, mul2(bc2(f.decay), w));
}

// structure kinds (FamilyScalars::kind), set by the host from the family and the step
enum : int { FK_PLAIN = 0,      // no state: SGD
             FK_M = 1,          // momentum-like state, linear direction: momentum / Nesterov
             FK_LION = 2,       // momentum-like state, sign direction
             FK_V = 3,          // second-moment state only: RMSprop, Adagrad
             FK_MV = 4,         // both, sqrt denominator: NAdam, rectified RAdam
             FK_MV_NODENOM = 5, // both, no denominator: RAdam while rho_t <= 5
             FK_MV_MAX = 6 };   // both, infinity norm: Adamax

}  // namespace forge
