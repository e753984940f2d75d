/*
 * forge_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU oracle for the
 * FORGE hot path (fused weight-gradient GEMM + AdamW), written from the paper.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no source, header, table or helper with the CUDA
 * path under paper_2606_22932_b200/csrc/ and includes nothing from include/.
 *
 * What it computes (Eq. 2-3; Eq. 4; Algorithm 1;
 * PAPER.md:253 "G_pq = sum_t dY_tp X_tq"; App. B for the int8 state):
 *
 *   g    = sum_{t=0}^{T-1} dY[t,p] * X[t,q]        bf16 inputs promoted to fp64, t ascending
 *   m'   = b1*m + (1-b1)*g                          Alg. 1 line 7
 *   v'   = b2*v + (1-b2)*g*g                        Alg. 1 line 8
 *   mhat = m'/(1-b1^t) ; vhat = v'/(1-b2^t)         Alg. 1 line 9
 *   W'   = (1-lr*wd)*W - lr*mhat/(sqrt(vhat)+eps)   Alg. 1 line 10
 *   store W' as bf16 (round to nearest even), m',v' in their storage type   Alg. 1 line 11
 *
 * Everything is fp64 until the final roundings.  Per Prop. 1 the tile-fused
 * schedule reaches exactly this result, so the oracle is the definition written out: form the
 * full G, then step every coordinate once.  No blocking, no fusion, no reordering.
 *
 * Readings of the paper where it is silent (listed in DESIGN.md "Readings"): S1 eps after the
 * sqrt of the bias-corrected v; S2 decay multiplies the pre-update W inside the same rounding;
 * S3 the W update uses the unrounded m',v'; S4 int8 blocks are 256 contiguous elements along
 * `in`; S5 m codes signed [-127,127] with scale a/127, v codes unsigned [0,255] with scale a/255,
 * the stored scale is the fp32 block absmax a; S6 nonzero-block v codes are floored at 1;
 * S7 rint (ties to even); S9 bf16 RNE straight from fp64; S10 step is 1-based; S15 the
 * hyper-parameters are the float values the ABI carries, promoted to double.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): exact rational brute force for g; closed form at
 * step 1 from zero state; torch.optim.AdamW in float64 for the general step; torch's fp32->bf16
 * cast for the rounding; App. B's s/2 bound, extremal codes and idempotence for the quantiser;
 * Prop. 1 (tile-by-tile == one shot, bit for bit).  Parity unpinned: the printed digits of
 * App. E -- inputs and hyper-parameters of that table are not given.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include <string.h>

/* ---------------------------------------------------------------- bf16 <-> fp64 ------------ */

/* bf16 bit pattern -> double (exact: bf16 is the top half of an IEEE binary32). */
double forge_oracle_bf16_to_double(uint16_t h)
{
    uint32_t u = ((uint32_t)h) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* double -> bf16, round to nearest, ties to even, in ONE rounding (no fp32 intermediate).
 * bf16: 1 sign, 8 exponent (bias 127), 7 fraction bits.  PAPER.md:1292-1293 names RNE for the
 * plain bf16 store.  NaN stays NaN, overflow goes to +-Inf. */
uint16_t forge_oracle_bf16_from_double(double x)
{
    uint16_t sign = signbit(x) ? 0x8000u : 0u;
    if (isnan(x)) return (uint16_t)(sign | 0x7FC0u);
    double a = fabs(x);
    if (isinf(a)) return (uint16_t)(sign | 0x7F80u);
    if (a == 0.0) return sign;

    int e;                               /* a = f * 2^e with f in [0.5,1)  =>  floor(log2 a) = e-1 */
    (void)frexp(a, &e);
    int p = e - 1;
    if (p < -126) p = -126;              /* subnormal range shares the ulp of the smallest normal */
    double ulp = ldexp(1.0, p - 7);      /* spacing of bf16 numbers in [2^p, 2^(p+1)) */
    double q = rint(a / ulp);            /* exact division by a power of two; rint = ties to even */
    double r = q * ulp;                  /* the rounded magnitude, exactly representable in fp32 */
    if (r >= ldexp(1.0, 128)) return (uint16_t)(sign | 0x7F80u);
    float rf = (float)r;                 /* exact */
    uint32_t u;
    memcpy(&u, &rf, sizeof u);
    return (uint16_t)(sign | (uint16_t)(u >> 16));
}

/* ---------------------------------------------------------------- the gradient ------------- */

/* G[p,q] = sum_t dY[t,p]*X[t,q], t ascending, fp64 (Eq. 3).
 * dY is [T,out] row-major with leading dimension lddy, X is [T,in] with ldx (elements).
 * If E != NULL it also receives sum_t |dY[t,p]|*|X[t,q]| (the magnitude sum the fp32
 * accumulation-error bound e_ij = T*2^-23*E_ij of BASELINE.json north_star is built on).
 * Rows p in [p0,p1) only: rows are independent, so a row subset is an exact oracle for them. */
void forge_oracle_wgrad_rows(const uint16_t *dY, const uint16_t *X, int T, int out, int in,
                             long lddy, long ldx, int p0, int p1, double *G, double *E)
{
    (void)out;
#pragma omp parallel for schedule(dynamic, 1)
    for (int p = p0; p < p1; ++p) {
        double *g = G + (size_t)(p - p0) * (size_t)in;
        double *e = E ? E + (size_t)(p - p0) * (size_t)in : NULL;
        for (int q = 0; q < in; ++q) g[q] = 0.0;
        if (e) for (int q = 0; q < in; ++q) e[q] = 0.0;
        for (int t = 0; t < T; ++t) {
            double dy = forge_oracle_bf16_to_double(dY[(size_t)t * (size_t)lddy + (size_t)p]);
            const uint16_t *xr = X + (size_t)t * (size_t)ldx;
            for (int q = 0; q < in; ++q) {
                double x = forge_oracle_bf16_to_double(xr[q]);
                g[q] += dy * x;
                if (e) e[q] += fabs(dy) * fabs(x);
            }
        }
    }
}

void forge_oracle_wgrad(const uint16_t *dY, const uint16_t *X, int T, int out, int in,
                        double *G, double *E)
{
    forge_oracle_wgrad_rows(dY, X, T, out, in, out, in, 0, out, G, E);
}

/* ---------------------------------------------------------------- AdamW, one coordinate ---- */

typedef struct {
    double lr, beta1, beta2, eps, wd;   /* the ABI's float values promoted to double (S15) */
    double bc1, bc2;                    /* 1-beta1^t, 1-beta2^t, t 1-based (S10) */
} forge_oracle_hp;

static forge_oracle_hp make_hp(long step, float lr, float beta1, float beta2, float eps, float wd)
{
    forge_oracle_hp h;
    h.lr = (double)lr; h.beta1 = (double)beta1; h.beta2 = (double)beta2;
    h.eps = (double)eps; h.wd = (double)wd;
    h.bc1 = 1.0 - pow(h.beta1, (double)step);
    h.bc2 = 1.0 - pow(h.beta2, (double)step);
    return h;
}

/* Algorithm 1 lines 7-10, one coordinate, fp64. */
static void adamw_coord(const forge_oracle_hp *h, double w, double m, double v, double g,
                        double *w_new, double *m_new, double *v_new)
{
    double m1 = h->beta1 * m + (1.0 - h->beta1) * g;                       /* line 7  */
    double v1 = h->beta2 * v + (1.0 - h->beta2) * g * g;                   /* line 8  */
    double mhat = m1 / h->bc1;                                             /* line 9  */
    double vhat = v1 / h->bc2;
    *w_new = (1.0 - h->lr * h->wd) * w - h->lr * mhat / (sqrt(vhat) + h->eps);  /* line 10 */
    *m_new = m1;
    *v_new = v1;
}

/* fp32 moments.  n = out*in coordinates; W bf16 bits, m, v fp32, all updated in place.
 * If Wd/md/vd != NULL they receive the unrounded fp64 results (used by tests for tolerances). */
void forge_oracle_adamw_fp32(uint16_t *W, float *m, float *v, const double *G, size_t n,
                             long step, float lr, float beta1, float beta2, float eps, float wd,
                             double *Wd, double *md, double *vd)
{
    forge_oracle_hp h = make_hp(step, lr, beta1, beta2, eps, wd);
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
        double w1, m1, v1;
        adamw_coord(&h, forge_oracle_bf16_to_double(W[i]), (double)m[i], (double)v[i], G[i],
                    &w1, &m1, &v1);
        W[i] = forge_oracle_bf16_from_double(w1);     /* line 11 */
        m[i] = (float)m1;                             /* fp64 -> fp32 RNE */
        v[i] = (float)v1;
        if (Wd) Wd[i] = w1;
        if (md) md[i] = m1;
        if (vd) vd[i] = v1;
    }
}

/* bf16 moments (the paper's "bf16-state" recipe): same update, m and v
 * stored bf16 RNE; W' is computed from the unrounded m', v' (reading S3). */
void forge_oracle_adamw_bf16(uint16_t *W, uint16_t *m, uint16_t *v, const double *G, size_t n,
                             long step, float lr, float beta1, float beta2, float eps, float wd,
                             double *Wd, double *md, double *vd)
{
    forge_oracle_hp h = make_hp(step, lr, beta1, beta2, eps, wd);
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
        double w1, m1, v1;
        adamw_coord(&h, forge_oracle_bf16_to_double(W[i]), forge_oracle_bf16_to_double(m[i]),
                    forge_oracle_bf16_to_double(v[i]), G[i], &w1, &m1, &v1);
        W[i] = forge_oracle_bf16_from_double(w1);
        m[i] = forge_oracle_bf16_from_double(m1);
        v[i] = forge_oracle_bf16_from_double(v1);
        if (Wd) Wd[i] = w1;
        if (md) md[i] = m1;
        if (vd) vd[i] = v1;
    }
}

/* ---------------------------------------------------------------- int8 blockwise state ----- */

#define FORGE_ORACLE_QBLOCK 256   /* BASELINE.json: 256-element blocks along `in` (reading S4) */

/* App. B: "m blockwise symmetric int8 ... a block with absolute maximum a has scale
 * s = a/127 and round-to-nearest quantization q(x) = s*round(x/s)".  Written out in fp64 from the fp64
 * moments: a = max|x| over the block, stored as fp32 (north_star: "fp32 absmax scale"); s = a/127 with
 * that stored a; code = rint(x/s) (S7: ties to even), clamped to [-127,127] (the fp32 rounding of a can
 * put |x/s| a hair above 127).  An all-zero block stores a = 0 and codes 0. */
void forge_oracle_quant_m_block(const double *x, int n, int8_t *code, float *scale)
{
    double amax = 0.0;
    for (int i = 0; i < n; ++i) { double f = fabs(x[i]); if (f > amax) amax = f; }
    float a = (float)amax;
    *scale = a;
    if (!(a > 0.0f)) { for (int i = 0; i < n; ++i) code[i] = 0; return; }
    double s = (double)a / 127.0;
    for (int i = 0; i < n; ++i) {
        double r = rint(x[i] / s);
        if (r > 127.0) r = 127.0;
        if (r < -127.0) r = -127.0;
        code[i] = (int8_t)r;
    }
}

/* v >= 0: unsigned linear code in [0,255], s = a/255 (S5); "v is floored away from zero"
 * (PAPER.md:316): in a block with a > 0 every code is at least 1 (S6). */
void forge_oracle_quant_v_block(const double *x, int n, uint8_t *code, float *scale)
{
    double amax = 0.0;
    for (int i = 0; i < n; ++i) { double f = fabs(x[i]); if (f > amax) amax = f; }
    float a = (float)amax;
    *scale = a;
    if (!(a > 0.0f)) { for (int i = 0; i < n; ++i) code[i] = 0; return; }
    double s = (double)a / 255.0;
    for (int i = 0; i < n; ++i) {
        double r = rint(x[i] / s);
        if (r > 255.0) r = 255.0;
        if (r < 1.0) r = 1.0;
        code[i] = (uint8_t)r;
    }
}

double forge_oracle_dequant_m(int8_t code, float scale)  { return (double)code * ((double)scale / 127.0); }
double forge_oracle_dequant_v(uint8_t code, float scale) { return (double)code * ((double)scale / 255.0); }

/* Quantise a whole [out,in] fp64 matrix row by row in blocks of 256 along `in` (in % 256 == 0).
 * Scales are [out, in/256] fp32. */
void forge_oracle_quant_matrix(const double *xm, const double *xv, int out, int in,
                               int8_t *mq, uint8_t *vq, float *m_scale, float *v_scale)
{
    int nb = in / FORGE_ORACLE_QBLOCK;
#pragma omp parallel for schedule(static)
    for (int p = 0; p < out; ++p)
        for (int b = 0; b < nb; ++b) {
            size_t o = (size_t)p * (size_t)in + (size_t)b * FORGE_ORACLE_QBLOCK;
            size_t s = (size_t)p * (size_t)nb + (size_t)b;
            if (xm) forge_oracle_quant_m_block(xm + o, FORGE_ORACLE_QBLOCK, mq + o, m_scale + s);
            if (xv) forge_oracle_quant_v_block(xv + o, FORGE_ORACLE_QBLOCK, vq + o, v_scale + s);
        }
}

/* int8 moments: dequantise, step in fp64 with the unrounded m',v' feeding W' (S3), requantise
 * every step with a fresh block absmax ("re-quantized every step"). */
void forge_oracle_adamw_int8(uint16_t *W, int8_t *mq, uint8_t *vq, float *m_scale, float *v_scale,
                             const double *G, int out, int in,
                             long step, float lr, float beta1, float beta2, float eps, float wd,
                             double *Wd, double *md, double *vd)
{
    forge_oracle_hp h = make_hp(step, lr, beta1, beta2, eps, wd);
    int nb = in / FORGE_ORACLE_QBLOCK;
#pragma omp parallel for schedule(static)
    for (int p = 0; p < out; ++p)
        for (int b = 0; b < nb; ++b) {
            double m1[FORGE_ORACLE_QBLOCK], v1[FORGE_ORACLE_QBLOCK];
            size_t o = (size_t)p * (size_t)in + (size_t)b * FORGE_ORACLE_QBLOCK;
            size_t s = (size_t)p * (size_t)nb + (size_t)b;
            for (int i = 0; i < FORGE_ORACLE_QBLOCK; ++i) {
                double w1;
                adamw_coord(&h, forge_oracle_bf16_to_double(W[o + i]),
                            forge_oracle_dequant_m(mq[o + i], m_scale[s]),
                            forge_oracle_dequant_v(vq[o + i], v_scale[s]),
                            G[o + i], &w1, &m1[i], &v1[i]);
                W[o + i] = forge_oracle_bf16_from_double(w1);
                if (Wd) Wd[o + i] = w1;
                if (md) md[o + i] = m1[i];
                if (vd) vd[o + i] = v1[i];
            }
            forge_oracle_quant_m_block(m1, FORGE_ORACLE_QBLOCK, mq + o, m_scale + s);
            forge_oracle_quant_v_block(v1, FORGE_ORACLE_QBLOCK, vq + o, v_scale + s);
        }
}

/* Array helper for tests: y[i] = bf16_RNE(x[i]). */
void forge_oracle_bf16_from_double_array(const double *x, uint16_t *y, size_t n)
{
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) y[i] = forge_oracle_bf16_from_double(x[i]);
}

int forge_oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = __builtin_omp_get_num_threads();
    }
#endif
    return n;
}
