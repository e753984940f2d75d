/* TEST INFRASTRUCTURE ONLY -- CPU oracle for the other coordinate-wise ("regime 1", tile-local A and U)
 * optimizer families of PAPER.md:267 Definition 1 / PAPER.md:716-727 Appendix I: SGD, SGD with momentum
 * (optionally Nesterov), Lion, RMSprop, Adagrad, Adamax, NAdam, RAdam.  The paper gives no formulas for
 * them: it verifies each "against a reference PyTorch implementation", so each function
 * below is the textbook rule as torch.optim documents it (Lion: Chen et al. 2023, Alg. 2), written out
 * per coordinate in fp64, one rounding to the storage type at the end, W' from the unrounded new state
 * (reading S3).  Pinned in tests/test_oracle_families.py against torch.optim in float64.
 * Shares nothing with the CUDA path.
 *
 * Hyper-parameters arrive as the ABI's floats and are promoted to double (reading S15).
 * State tensors: s0 / s1, fp32 or bf16 bit patterns (state_bf16 != 0); absent ones are NULL.
 *   SGD        : no state            MOMENTUM : s0 = momentum buffer    LION    : s0 = m
 *   RMSPROP    : s0 = square avg     ADAGRAD  : s0 = sum of squares
 *   ADAMAX     : s0 = m, s1 = u (infinity norm)     NADAM, RADAM : s0 = m, s1 = v
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

double forge_oracle_bf16_to_double(uint16_t b);
uint16_t forge_oracle_bf16_from_double(double x);

enum { FAM_SGD = 1, FAM_MOMENTUM = 2, FAM_LION = 3, FAM_RMSPROP = 4, FAM_ADAGRAD = 5, FAM_ADAMAX = 6,
       FAM_NADAM = 7, FAM_RADAM = 8 };

typedef struct {
    int family;
    long step;                 /* 1-based index of the update being applied */
    double lr, beta1, beta2, eps, wd;
    double momentum;           /* MOMENTUM: mu; RMSPROP: alpha is passed in beta2 */
    int nesterov;
} fam_hp;

static double ld(const void *p, size_t i, int bf16)
{
    return bf16 ? forge_oracle_bf16_to_double(((const uint16_t *)p)[i]) : (double)((const float *)p)[i];
}
static void st(void *p, size_t i, int bf16, double x)
{
    if (bf16) ((uint16_t *)p)[i] = forge_oracle_bf16_from_double(x);
    else ((float *)p)[i] = (float)x;
}

/* NAdam's momentum schedule (torch.optim.NAdam, momentum_decay psi = 4e-3):
 * mu_t = beta1 * (1 - 0.5 * 0.96^(t*psi)); mu_product_t = prod_{i<=t} mu_i. */
static double nadam_mu(double beta1, long t) { return beta1 * (1.0 - 0.5 * pow(0.96, (double)t * 4e-3)); }

/* One coordinate.  w, s0, s1: current values; g: this step's gradient. */
static void family_coord(const fam_hp *h, double w, double s0, double s1, double g,
                         double *w1, double *s0n, double *s1n)
{
    const double t = (double)h->step;
    *s0n = s0; *s1n = s1;
    switch (h->family) {
    case FAM_SGD: {                                   /* torch.optim.SGD, momentum = 0 */
        double gp = g + h->wd * w;                    /* L2 (coupled) weight decay */
        *w1 = w - h->lr * gp;
        break; }
    case FAM_MOMENTUM: {                              /* torch.optim.SGD, dampening = 0 */
        double gp = g + h->wd * w;
        double buf = (h->step == 1) ? gp : h->momentum * s0 + gp;   /* first step: buf = g */
        double d = h->nesterov ? gp + h->momentum * buf : buf;
        *w1 = w - h->lr * d;
        *s0n = buf;
        break; }
    case FAM_LION: {                                  /* Chen et al. 2023, Algorithm 2 */
        double c = h->beta1 * s0 + (1.0 - h->beta1) * g;
        double sgn = (c > 0.0) - (c < 0.0);
        *w1 = w * (1.0 - h->lr * h->wd) - h->lr * sgn;             /* decoupled decay */
        *s0n = h->beta2 * s0 + (1.0 - h->beta2) * g;
        break; }
    case FAM_RMSPROP: {                               /* torch.optim.RMSprop, momentum 0, not centered */
        double gp = g + h->wd * w;
        double sq = h->beta2 * s0 + (1.0 - h->beta2) * gp * gp;    /* alpha passed as beta2 */
        *w1 = w - h->lr * gp / (sqrt(sq) + h->eps);
        *s0n = sq;
        break; }
    case FAM_ADAGRAD: {                               /* torch.optim.Adagrad, lr_decay = 0 */
        double gp = g + h->wd * w;
        double sum = s0 + gp * gp;
        *w1 = w - h->lr * gp / (sqrt(sum) + h->eps);
        *s0n = sum;
        break; }
    case FAM_ADAMAX: {                                /* torch.optim.Adamax */
        double gp = g + h->wd * w;
        double m = h->beta1 * s0 + (1.0 - h->beta1) * gp;
        double u = fmax(h->beta2 * s1, fabs(gp) + h->eps);
        *w1 = w - (h->lr / (1.0 - pow(h->beta1, t))) * m / u;
        *s0n = m; *s1n = u;
        break; }
    case FAM_NADAM: {                                 /* torch.optim.NAdam, coupled decay */
        double gp = g + h->wd * w;
        double bc2 = 1.0 - pow(h->beta2, t);
        double mu = nadam_mu(h->beta1, h->step), mu_next = nadam_mu(h->beta1, h->step + 1);
        double prod = 1.0;
        for (long i = 1; i <= h->step; ++i) prod *= nadam_mu(h->beta1, i);
        double m = h->beta1 * s0 + (1.0 - h->beta1) * gp;
        double v = h->beta2 * s1 + (1.0 - h->beta2) * gp * gp;
        double denom = sqrt(v / bc2) + h->eps;
        *w1 = w - h->lr * (1.0 - mu) / (1.0 - prod) * gp / denom
                - h->lr * mu_next / (1.0 - prod * mu_next) * m / denom;
        *s0n = m; *s1n = v;
        break; }
    case FAM_RADAM: {                                 /* torch.optim.RAdam, coupled decay */
        double gp = g + h->wd * w;
        double bc1 = 1.0 - pow(h->beta1, t), bc2 = 1.0 - pow(h->beta2, t);
        double m = h->beta1 * s0 + (1.0 - h->beta1) * gp;
        double v = h->beta2 * s1 + (1.0 - h->beta2) * gp * gp;
        double rho_inf = 2.0 / (1.0 - h->beta2) - 1.0;
        double rho_t = rho_inf - 2.0 * t * pow(h->beta2, t) / bc2;
        double mhat = m / bc1;
        if (rho_t > 5.0) {
            double rect = sqrt((rho_t - 4.0) * (rho_t - 2.0) * rho_inf / ((rho_inf - 4.0) * (rho_inf - 2.0) * rho_t));
            double adaptive = sqrt(bc2) / (sqrt(v) + h->eps);
            *w1 = w - mhat * h->lr * adaptive * rect;
        } else {
            *w1 = w - mhat * h->lr;
        }
        *s0n = m; *s1n = v;
        break; }
    default:
        *w1 = w;
    }
}

/* n coordinates, in place.  W bf16 bits; s0/s1 fp32 or bf16 bits (NULL when the family has none).
 * Wd (optional) receives the unrounded fp64 W'. */
void forge_oracle_family_step(int family, uint16_t *W, void *s0, void *s1, int state_bf16, const double *G,
                              size_t n, long step, float lr, float beta1, float beta2, float eps, float wd,
                              float momentum, int nesterov, double *Wd)
{
    fam_hp h;
    h.family = family; h.step = step; h.lr = (double)lr; h.beta1 = (double)beta1; h.beta2 = (double)beta2;
    h.eps = (double)eps; h.wd = (double)wd; h.momentum = (double)momentum; h.nesterov = nesterov;
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
        double w1, a, b;
        family_coord(&h, forge_oracle_bf16_to_double(W[i]), s0 ? ld(s0, i, state_bf16) : 0.0,
                     s1 ? ld(s1, i, state_bf16) : 0.0, G[i], &w1, &a, &b);
        W[i] = forge_oracle_bf16_from_double(w1);
        if (s0) st(s0, i, state_bf16, a);
        if (s1) st(s1, i, state_bf16, b);
        if (Wd) Wd[i] = w1;
    }
}

/* Accumulate-into-state, the paper's regime 2 ("B <- mu B + G is tile-local and affine, so the
 * weight-gradient multiply accumulates in place into the momentum buffer through the GEMM's own beta";
 * PAPER.md:757-759 Muon's A-step).  Per coordinate in fp64, one rounding to the storage type. */
void forge_oracle_accumulate(void *B, int state_bf16, const double *G, size_t n, float mu)
{
    const double m = (double)mu;
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) st(B, i, state_bf16, m * ld(B, i, state_bf16) + G[i]);
}

/* ---------------------------------------------------------------- stochastic-rounding store --
 * The paper's "SR-store" recipe (1287-1296: "the bf16 weight is the only copy, committed by
 * stochastic rounding"; microcheck PAPER.md:1450 "dead zone, unbiasedness").  The paper gives no generator,
 * so both sides implement the same counter-based one (reading S16): 16 random bits r16 per weight
 * element from (seed, step, stream, row, col) through the murmur3 finaliser, u = r16 / 65536 uniform on [0,1).
 * The rounding itself is the textbook rule on the fp64 value W': with lo, hi its two bf16 neighbours (lo toward
 * zero) and frac = (|W'| - lo) / (hi - lo), the store takes hi iff u >= 1 - frac, i.e. with probability frac
 * (to the 2^-16 resolution of u) -- unbiased.  Inf / NaN take the RNE path. */
static uint32_t fmix32(uint32_t h)
{
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    return h;
}
uint32_t forge_oracle_sr_bits(uint64_t seed, long step, uint32_t stream, uint32_t row, uint32_t col)
{
    uint32_t inner = fmix32((uint32_t)(seed >> 32) ^ ((uint32_t)step * 0x85EBCA77u) ^ (stream * 0xC2B2AE3Du));
    uint32_t rowkey = fmix32((row * 0x9E3779B1u) ^ (uint32_t)seed ^ inner);
    return fmix32(rowkey ^ (col * 0x27D4EB2Fu)) >> 16;
}
uint16_t forge_oracle_bf16_sr_from_double(double x, uint32_t r16)
{
    if (isnan(x) || isinf(x) || x == 0.0) return forge_oracle_bf16_from_double(x);
    uint16_t sign = signbit(x) ? 0x8000u : 0u;
    double a = fabs(x);
    int e;
    (void)frexp(a, &e);
    int p = e - 1;
    if (p < -126) p = -126;
    double ulp = ldexp(1.0, p - 7);                        /* spacing of bf16 numbers around |x| */
    double q = a / ulp;                                   /* exact (power of two) */
    double fl = floor(q), frac = q - fl;                  /* exact */
    if ((double)r16 + frac * 65536.0 >= 65536.0) fl += 1.0;
    double r = fl * ulp;
    if (r >= ldexp(1.0, 128)) return (uint16_t)(sign | 0x7F80u);
    float rf = (float)r;                                  /* exact: r is a bf16 value */
    uint32_t b;
    __builtin_memcpy(&b, &rf, 4);
    return (uint16_t)(sign | (uint16_t)(b >> 16));
}

/* AdamW (Algorithm 1) with fp32 moments and the SR store of W; W is [out, in]. */
void forge_oracle_adamw_fp32_sr(uint16_t *W, float *m, float *v, const double *G, int out, int in, long step,
                                float lr, float beta1, float beta2, float eps, float wd, uint64_t seed, uint32_t stream)
{
    const double b1 = beta1, b2 = beta2, bc1 = 1.0 - pow(b1, (double)step), bc2 = 1.0 - pow(b2, (double)step);
#pragma omp parallel for schedule(static)
    for (int p = 0; p < out; ++p)
        for (int q = 0; q < in; ++q) {
            size_t i = (size_t)p * in + q;
            double w = forge_oracle_bf16_to_double(W[i]);
            double m1 = b1 * (double)m[i] + (1.0 - b1) * G[i];
            double v1 = b2 * (double)v[i] + (1.0 - b2) * G[i] * G[i];
            double w1 = (1.0 - (double)lr * (double)wd) * w - (double)lr * (m1 / bc1) / (sqrt(v1 / bc2) + (double)eps);
            W[i] = forge_oracle_bf16_sr_from_double(w1, forge_oracle_sr_bits(seed, step, stream, (uint32_t)p, (uint32_t)q));
            m[i] = (float)m1;
            v[i] = (float)v1;
        }
}

/* ---------------------------------------------------------------- fp8 moments ---------------
 * "FORGE fp8 states (per-tensor scale) ... per-tensor scaled with delayed scaling, so its error is reported
 * rather than bounded".  The paper fixes neither the format nor the scaling rule; DESIGN.md
 * reading S17: m and v are stored as e4m3 (4 exponent bits, bias 7, 3 mantissa bits, max finite 448, no Inf)
 * codes of x / s with one fp32 scale s per tensor; DELAYED scaling: the scale in use was derived by the caller
 * from the amax the previous step reported (s = amax_prev / 448); this step reports its own amax of m', v'
 * for the next one.  Values beyond 448 s saturate (round-to-nearest-even, satfinite -- the hardware cvt).
 * code = e4m3(x / s) evaluated in fp64 from the fp64 moment and the stored fp32 scale; s = 0 stores code 0. */
uint8_t forge_oracle_e4m3_from_double(double t)
{
    uint8_t sign = signbit(t) ? 0x80u : 0u;
    double a = fabs(t);
    if (t != t) return (uint8_t)(sign | 0x7Fu);            /* NaN */
    if (a > 448.0) return (uint8_t)(sign | 0x7Eu);         /* satfinite (includes Inf) */
    if (a < 0.015625) {                                    /* below the smallest normal 2^-6: subnormal grid 2^-9 */
        int q = (int)rint(a * 512.0);                      /* ties to even; q == 8 is the smallest normal, code 0x08 */
        return (uint8_t)(sign | (uint8_t)q);
    }
    int e;
    double f = frexp(a, &e);                               /* a = f * 2^e, f in [0.5, 1) */
    double mant = f * 2.0; e -= 1;                         /* mant in [1, 2) */
    int q = (int)rint((mant - 1.0) * 8.0);
    if (q == 8) { q = 0; e += 1; }
    int code = ((e + 7) << 3) | q;
    if (code > 0x7E) code = 0x7E;
    return (uint8_t)(sign | (uint8_t)code);
}
uint8_t forge_oracle_e4m3_from_float(float t) { return forge_oracle_e4m3_from_double((double)t); }
double forge_oracle_e4m3_to_double(uint8_t c)
{
    double s = (c & 0x80u) ? -1.0 : 1.0;
    int e = (c >> 3) & 0xF, q = c & 7;
    if (e == 0xF && q == 7) return NAN;
    if (e == 0) return s * (double)q * 0.001953125;        /* q * 2^-9 */
    return s * (1.0 + (double)q / 8.0) * ldexp(1.0, e - 7);
}
static double fp8_scaled(double x, float s) { return s > 0.0f ? x / (double)s : 0.0; }

/* quantise one fp32 tensor: scale = amax / 448 stored as fp32, codes as above */
void forge_oracle_fp8_quantize(const float *x, size_t n, uint8_t *code, float *scale)
{
    double amax = 0.0;
    for (size_t i = 0; i < n; ++i) { double a = fabs((double)x[i]); if (a > amax) amax = a; }
    float s = (float)(amax / 448.0);
    *scale = s;
    for (size_t i = 0; i < n; ++i) code[i] = forge_oracle_e4m3_from_double(fp8_scaled((double)x[i], s));
}

/* AdamW (Algorithm 1) with e4m3 moments.  m_scale / v_scale: [0] = scale in use (read),
 * [1] = amax of this step's m' / v' (max-accumulated into the incoming value). */
void forge_oracle_adamw_fp8(uint16_t *W, uint8_t *mq, uint8_t *vq, float *m_scale, float *v_scale, const double *G,
                            size_t n, long step, float lr, float beta1, float beta2, float eps, float wd)
{
    const double b1 = beta1, b2 = beta2, bc1 = 1.0 - pow(b1, (double)step), bc2 = 1.0 - pow(b2, (double)step);
    const double sm = (double)m_scale[0], sv = (double)v_scale[0];
    float am = m_scale[1], av = v_scale[1];
#pragma omp parallel for schedule(static) reduction(max : am, av)
    for (size_t i = 0; i < n; ++i) {
        double w = forge_oracle_bf16_to_double(W[i]);
        double m1 = b1 * (forge_oracle_e4m3_to_double(mq[i]) * sm) + (1.0 - b1) * G[i];
        double v1 = b2 * (forge_oracle_e4m3_to_double(vq[i]) * sv) + (1.0 - b2) * G[i] * G[i];
        double w1 = (1.0 - (double)lr * (double)wd) * w - (double)lr * (m1 / bc1) / (sqrt(v1 / bc2) + (double)eps);
        W[i] = forge_oracle_bf16_from_double(w1);
        mq[i] = forge_oracle_e4m3_from_double(fp8_scaled(m1, m_scale[0]));
        vq[i] = forge_oracle_e4m3_from_double(fp8_scaled(v1, v_scale[0]));
        float fm = fabsf((float)m1), fv = fabsf((float)v1);
        if (fm > am) am = fm;
        if (fv > av) av = fv;
    }
    m_scale[1] = am;
    v_scale[1] = av;
}
