/*
 * aria_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU definition of the quantized DiT linear
 * layers (W8A8 and W4A16) of arxiv/paper_2607_08526 ("aria").  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may build, load or call this file.  It shares no code, header, table or
 * constant with paper_2607_08526_b200/csrc (the CUDA path).
 *
 * What the paper fixes: PAPER.md L78 (SIII-A(b)): DiT weights "compressed to
 * 8-bit or 4-bit integers (q8, q4)"; "an optional mode also runs the arithmetic
 * in 8-bit, quantizing activations alongside weights (W8A8)".  The paper fixes
 * NO scheme (granularity, rounding, scale dtype), so the schemes are the ones
 * BASELINE.json `configs` C1-C5 state, read as SURVEY.md S8(c) O1-O5 / DESIGN.md
 * "Readings" R1-R17.  Each function cites the reading it follows.
 *
 * Arithmetic rules: scalar loops, one IEEE operation per C expression where the
 * definition names an fp32 rounding (build with -ffp-contract=off, no
 * -ffast-math), int64 accumulation for int8 products, fp64 accumulation for
 * bf16 products.  OpenMP, when enabled, splits rows only; every row is computed
 * by exactly the same scalar code, so results do not depend on thread count.
 *
 * Parity pins: tests/test_oracle_*.py (hand-worked H1/H2 from SURVEY.md S8(c),
 * brute-force nearest-code search, invariants, closed forms, numpy fp64 matmul,
 * numpy/ml_dtypes conversions; O6 and O7: hand-worked H3 / H4 in tests/golden/,
 * integer special cases, numpy, the alpha = 0 / beta = -1 invariants; O8 and O9:
 * hand-worked H5 / H6 in tests/golden/, zero-mean / unit-variance and shift / scale
 * invariances, uniform and one-hot attention, key-permutation and key-shift
 * invariance, torch fp64 layer_norm / scaled_dot_product_attention as the library
 * routine).
 * Parity unpinned: none.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* ---------------------------------------------------------------- helpers */

/* bf16 bit pattern -> fp32 (exact: bf16 is the top 16 bits of an fp32). */
float oracle_bf16_bits_to_f32(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}

/* fp16 bit pattern -> fp32 (exact), written out from the IEEE-754 binary16
 * definition: 1 sign, 5 exponent (bias 15), 10 fraction bits. */
float oracle_fp16_bits_to_f32(uint16_t h)
{
    int sign = (h >> 15) & 1;
    int e = (h >> 10) & 0x1F;
    int f = h & 0x3FF;
    double v;
    if (e == 0)
        v = ldexp((double)f, -24); /* subnormal: f * 2^-24 */
    else if (e == 31)
        v = f ? NAN : INFINITY;
    else
        v = ldexp(1.0 + (double)f / 1024.0, e - 15);
    return (float)(sign ? -v : v);
}

/* Round a finite double to the nearest value with `p` significand bits and
 * minimum normal exponent `emin` (value = m * 2^e, 1 <= m < 2, e >= emin;
 * below that the spacing is fixed at 2^(emin-p+1): gradual underflow), ties to
 * even.  rint() rounds half to even in the default rounding mode.  Overflow
 * beyond `emax` returns +-inf.  This is IEEE round-to-nearest-even written
 * out; it is used for fp16 (p=11, emin=-14, emax=15) and bf16 (p=8, emin=-126,
 * emax=127). */
static double round_to_format(double x, int p, int emin, int emax)
{
    if (x == 0.0 || isnan(x) || isinf(x))
        return x;
    int e;
    (void)frexp(fabs(x), &e); /* |x| = m * 2^e, 0.5 <= m < 1  => exponent e-1 */
    int ex = e - 1;
    if (ex < emin)
        ex = emin;
    double quantum = ldexp(1.0, ex - (p - 1));
    double r = rint(x / quantum) * quantum; /* x/quantum is exact (power of 2) */
    if (fabs(r) >= ldexp(1.0, emax + 1))
        return x > 0 ? INFINITY : -INFINITY;
    return r;
}

/* fp32 -> fp16 bits, round-to-nearest-even, subnormals kept (reading R7). */
uint16_t oracle_f32_to_fp16_bits(float x)
{
    uint16_t sign = signbit(x) ? 0x8000 : 0;
    if (isnan(x))
        return (uint16_t)(sign | 0x7E00);
    double r = fabs(round_to_format((double)x, 11, -14, 15));
    if (isinf(r))
        return (uint16_t)(sign | 0x7C00);
    if (r == 0.0)
        return sign;
    if (r < ldexp(1.0, -14)) /* subnormal: r = f * 2^-24 */
        return (uint16_t)(sign | (uint16_t)(r * 16777216.0));
    int e;
    double m = frexp(r, &e); /* r = m*2^e, m in [0.5,1) -> 1.f * 2^(e-1) */
    int f = (int)((m * 2.0 - 1.0) * 1024.0);
    return (uint16_t)(sign | ((e - 1 + 15) << 10) | f);
}

/* double -> bf16 bits with ONE rounding (no detour through fp32). */
uint16_t oracle_f64_to_bf16_bits(double x)
{
    uint16_t sign = signbit(x) ? 0x8000 : 0;
    if (isnan(x))
        return (uint16_t)(sign | 0x7FC0);
    double r = fabs(round_to_format(x, 8, -126, 127));
    if (isinf(r))
        return (uint16_t)(sign | 0x7F80);
    float f = (float)r; /* exact: r has 8 significant bits in fp32 range */
    uint32_t u;
    memcpy(&u, &f, 4);
    return (uint16_t)(sign | (u >> 16));
}

/* exact-erf GELU in fp64 (reading R11): gelu(y) = 0.5*y*(1+erf(y/sqrt 2)). */
double oracle_gelu_erf(double y)
{
    return 0.5 * y * (1.0 + erf(y / sqrt(2.0)));
}

/* round-half-to-even of an fp32 value to an int, then clamp to [-lim, lim]. */
static int rint_clamp(float v, int lim)
{
    float r = rintf(v); /* default rounding mode: ties to even */
    int q = (int)r;
    if (q > lim)
        q = lim;
    if (q < -lim)
        q = -lim;
    return q;
}

/* -------------------------------------------------------------------- O1 */
/* Per-row symmetric int8 quantisation (configs C1-C3:
 * "scale=absmax/127, round-half-even, clamp +-127"; readings R2-R4).
 *   a = max_c |A[r,c]|            (exact)
 *   s = a > 0 ? fl32(a / 127) : 1
 *   q = clamp(rint(fl32(A[r,c] / s)), -127, 127)
 * Used for activations (row = token) and for int8 weights (row = output
 * channel).  A is fp32 (bf16 inputs are widened exactly by the caller). */
void oracle_quant_int8_rows(const float *A, int64_t R, int64_t C, int8_t *q, float *s)
{
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < R; ++r) {
        const float *row = A + r * C;
        float a = 0.0f;
        for (int64_t c = 0; c < C; ++c) {
            float v = fabsf(row[c]);
            if (v > a)
                a = v;
        }
        float sc = 1.0f;
        if (a > 0.0f)
            sc = a / 127.0f; /* one fp32 division */
        s[r] = sc;
        for (int64_t c = 0; c < C; ++c) {
            float t = row[c] / sc; /* one fp32 division */
            q[r * C + c] = (int8_t)rint_clamp(t, 127);
        }
    }
}

/* -------------------------------------------------------------------- O2 */
/* Group-wise symmetric int4 quantisation along K (config C4:
 * "symmetric int4 codes in [-7,7], group 32 along K, fp16 per-group scales, two
 * codes per byte"; readings R3, R4, R7, R8).
 *   a  = max |w| over the group
 *   sg = fp16_rne(fl32(a / 7))      (subnormals kept)
 *   sg == 0 -> codes 0;  else q = clamp(rint(fl32(w / float(sg))), -7, 7)
 * codes[N,K] int8 (unpacked, for tests); sg_bits[N,K/G] fp16 bit patterns;
 * packed[N,K/2]: byte j = (code[2j] & 0xF) | ((code[2j+1] & 0xF) << 4),
 * 4-bit two's complement. */
void oracle_quant_int4_groups(const float *W, int64_t N, int64_t K, int G, int8_t *codes,
                              uint16_t *sg_bits, uint8_t *packed)
{
    int64_t ng = K / G;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        for (int64_t g = 0; g < ng; ++g) {
            const float *w = W + n * K + g * G;
            float a = 0.0f;
            for (int i = 0; i < G; ++i) {
                float v = fabsf(w[i]);
                if (v > a)
                    a = v;
            }
            float s32 = a / 7.0f;
            uint16_t hb = oracle_f32_to_fp16_bits(s32);
            float sg = oracle_fp16_bits_to_f32(hb);
            sg_bits[n * ng + g] = hb;
            for (int i = 0; i < G; ++i) {
                int q = 0;
                if (sg != 0.0f) {
                    float t = w[i] / sg;
                    q = rint_clamp(t, 7);
                }
                codes[n * K + g * G + i] = (int8_t)q;
            }
        }
        for (int64_t j = 0; j < K / 2; ++j) {
            int lo = codes[n * K + 2 * j] & 0xF;
            int hi = codes[n * K + 2 * j + 1] & 0xF;
            packed[n * (K / 2) + j] = (uint8_t)(lo | (hi << 4));
        }
    }
}

/* Unpack the canonical int4 byte format back to codes (sign-extend nibbles). */
void oracle_unpack_int4(const uint8_t *packed, int64_t N, int64_t K, int8_t *codes)
{
    for (int64_t n = 0; n < N; ++n)
        for (int64_t j = 0; j < K / 2; ++j) {
            uint8_t b = packed[n * (K / 2) + j];
            int lo = b & 0xF, hi = (b >> 4) & 0xF;
            codes[n * K + 2 * j] = (int8_t)(lo >= 8 ? lo - 16 : lo);
            codes[n * K + 2 * j + 1] = (int8_t)(hi >= 8 ? hi - 16 : hi);
        }
}

/* -------------------------------------------------------------------- O3 */
/* int8 x int8 GEMM, exact: acc[m,n] = sum_k Xq[m,k] * Wq[n,k] in int64
 * (north_star "accumulates int8 products in int64").
 * Returns the number of entries that do not fit int32 (must be 0). */
int64_t oracle_gemm_i8(const int8_t *Xq, const int8_t *Wq, int64_t M, int64_t N, int64_t K,
                       int64_t *acc)
{
    int64_t overflow = 0;
#pragma omp parallel for schedule(static) reduction(+ : overflow)
    for (int64_t m = 0; m < M; ++m)
        for (int64_t n = 0; n < N; ++n) {
            int64_t a = 0;
            for (int64_t k = 0; k < K; ++k)
                a += (int64_t)Xq[m * K + k] * (int64_t)Wq[n * K + k];
            acc[m * N + n] = a;
            if (a > 2147483647LL || a < -2147483648LL)
                overflow += 1;
        }
    return overflow;
}

/* Rescale + bias (+ GELU) epilogue in fp64:
 *   y = (double)acc * (double)sx[m] * (double)sw[n] + (double)b[n]
 *   act == 1: y = gelu_erf(y)
 * bias may be NULL.  Output is fp64; rounding to the output dtype is a
 * separate, single step (oracle_round_out). */
void oracle_epilogue_w8a8(const int64_t *acc, const float *sx, const float *sw, const double *bias,
                          int act, int64_t M, int64_t N, double *y)
{
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < M; ++m)
        for (int64_t n = 0; n < N; ++n) {
            double v = (double)acc[m * N + n] * (double)sx[m] * (double)sw[n];
            if (bias)
                v += bias[n];
            if (act == 1)
                v = oracle_gelu_erf(v);
            y[m * N + n] = v;
        }
}

/* -------------------------------------------------------------------- O4 */
/* W4A16 linear (config C4; readings R12):
 *   variant 0: w^ = bf16_rne(float(q) * float(sg))   (product exact in fp32)
 *   variant 1: w^ = q * sg  exactly (not rounded to bf16)
 *   y = sum_k (double)x[m,k] * (double)w^[n,k] + (double)b[n]  (fp64)
 * X is fp32 holding bf16 values exactly.  codes[N,K] int8, sg_bits[N,K/G].
 * (Models of a kernel's operand FORMAT -- the former variants 2 and 3 -- are not definitions
 * and live with the tests: tests/kernel_models.py.) */

void oracle_linear_w4a16(const float *X, const int8_t *codes, const uint16_t *sg_bits,
                         const double *bias, int act, int variant, int64_t M, int64_t N,
                         int64_t K, int G, double *y)
{
    int64_t ng = K / G;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        double wrow[K];
        for (int64_t k = 0; k < K; ++k) {
            float sg = oracle_fp16_bits_to_f32(sg_bits[n * ng + k / G]);
            float prod = (float)codes[n * K + k] * sg; /* exact: 3-bit x 11-bit */
            if (variant == 0)
                wrow[k] = (double)oracle_bf16_bits_to_f32(oracle_f64_to_bf16_bits((double)prod));
            else
                wrow[k] = (double)prod;
        }
        for (int64_t m = 0; m < M; ++m) {
            double a = 0.0;
            for (int64_t k = 0; k < K; ++k)
                a += (double)X[m * K + k] * wrow[k];
            if (bias)
                a += bias[n];
            if (act == 1)
                a = oracle_gelu_erf(a);
            y[m * N + n] = a;
        }
    }
}

/* Dequantised weight matrix of variant 0/1 as fp64 [N,K] (for the pin that
 * reduces O4 to numpy.matmul). */
void oracle_dequant_int4(const int8_t *codes, const uint16_t *sg_bits, int variant, int64_t N,
                         int64_t K, int G, double *What)
{
    int64_t ng = K / G;
    for (int64_t n = 0; n < N; ++n)
        for (int64_t k = 0; k < K; ++k) {
            float sg = oracle_fp16_bits_to_f32(sg_bits[n * ng + k / G]);
            float prod = (float)codes[n * K + k] * sg;
            What[n * K + k] = variant == 0
                                  ? (double)oracle_bf16_bits_to_f32(oracle_f64_to_bf16_bits(prod))
                                  : (double)prod;
        }
}

/* -------------------------------------------------------------------- O6 */
/* q8 weight-only linear, "W8A16" (weights
 * "compressed to 8-bit ... integers (labelled q8)" with the arithmetic left in half
 * precision; Table II col. q8, L129-131).  Weights: the S0 int8 format (per-output-
 * channel scale sw[n], codes in [-127,127]); activations bf16; like O4 the
 * dequantised weight is fed to a bf16 GEMM with fp32 accumulation (R18):
 *   variant 0: w^ = bf16_rne(q * sw[n])   (ONE rounding of the exact product)
 *   variant 1: w^ = q * sw[n] exactly
 *   y = sum_k (double)x[m,k] * (double)w^[n,k] + (double)b[n]; act == 1: GELU. */
void oracle_linear_w8a16(const float *X, const int8_t *Wq, const float *sw, const double *bias,
                         int act, int variant, int64_t M, int64_t N, int64_t K, double *y)
{
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        double wrow[K];
        for (int64_t k = 0; k < K; ++k) {
            double prod = (double)Wq[n * K + k] * (double)sw[n]; /* exact: 8-bit x 24-bit */
            if (variant == 0)
                wrow[k] = (double)oracle_bf16_bits_to_f32(oracle_f64_to_bf16_bits(prod));
            else
                wrow[k] = prod;
        }
        for (int64_t m = 0; m < M; ++m) {
            double a = 0.0;
            for (int64_t k = 0; k < K; ++k)
                a += (double)X[m * K + k] * wrow[k];
            if (bias)
                a += bias[n];
            if (act == 1)
                a = oracle_gelu_erf(a);
            y[m * N + n] = a;
        }
    }
}

/* -------------------------------------------------------------------- O7 */
/* In-graph activation steering of the residual stream.
 * op 0, additive injection -- PAPER.md eq. 2 (L94-98): for every token row t
 *     h[t,:] <- h[t,:] + alpha * hbar_norm * d[:]
 *   "where ||h-bar|| is the mean baseline residual norm at l" (a given scalar),
 *   d the unit direction of eq. 1.
 * op 1, projection -- PAPER.md L192 / L248: "amplifying (beta > 0) or removing
 *   (beta < 0) the direction component already present per token":
 *     c_t = sum_j h[t,j] * d[j];   h[t,:] <- h[t,:] + beta * c_t * d[:]
 *   (beta = -1 removes the component when |d| = 1; R19).
 * Strength 0 "leaves the pass unchanged" (L98) / "the output is bit-identical to
 * the base model" (L77): the caller's array is returned untouched, -0.0 included.
 * All arithmetic in fp64; H is fp32 (bf16 values widened by the caller). */
void oracle_steer(const float *H, int64_t M, int64_t D, const float *d, double strength,
                  double hbar_norm, int op, double *out)
{
    for (int64_t t = 0; t < M; ++t) {
        double c = 0.0;
        if (op == 1)
            for (int64_t j = 0; j < D; ++j)
                c += (double)H[t * D + j] * (double)d[j];
        for (int64_t j = 0; j < D; ++j) {
            double h = (double)H[t * D + j];
            if (strength == 0.0)
                out[t * D + j] = h;
            else if (op == 0)
                out[t * D + j] = h + strength * hbar_norm * (double)d[j];
            else
                out[t * D + j] = h + strength * c * (double)d[j];
        }
    }
}

/* -------------------------------------------------------------------- O8 */
/* Normalisation that precedes QKV / MLP-up inside a DiT block, the producer whose
 * output S1 quantises (SURVEY S8(f) NEXT-2 "norm -> act-quant fusion"
 * names only "the diffusion transformer (DiT)" [10] and L224 / L278 the blocks'
 * self-attention; it gives no formula, so the textbook definitions are taken,
 * DESIGN.md R20):
 *   kind 0, LayerNorm:  mu = mean_k x;  var = mean_k (x - mu)^2  (biased);
 *                       n[k] = (x[k] - mu) / sqrt(var + eps) * gamma[k] + beta[k]
 *   kind 1, RMSNorm:    n[k] = x[k] / sqrt(mean_k x^2 + eps) * gamma[k] + beta[k]
 * beta may be NULL (0).  All arithmetic in fp64; the caller rounds n once to the
 * activation dtype (oracle_round_out) -- the tensor an unfused norm kernel would
 * store -- and feeds that to O1. */
void oracle_norm_rows(const float *X, int64_t M, int64_t K, const float *gamma, const float *beta,
                      int kind, double eps, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < M; ++m) {
        const float *x = X + m * K;
        double mu = 0.0;
        if (kind == 0) {
            for (int64_t k = 0; k < K; ++k)
                mu += (double)x[k];
            mu /= (double)K;
        }
        double var = 0.0;
        for (int64_t k = 0; k < K; ++k)
            var += ((double)x[k] - mu) * ((double)x[k] - mu);
        var /= (double)K;
        double rstd = 1.0 / sqrt(var + eps);
        for (int64_t k = 0; k < K; ++k)
            out[m * K + k] = ((double)x[k] - mu) * rstd * (double)gamma[k] + (beta ? (double)beta[k] : 0.0);
    }
}

/* -------------------------------------------------------------------- O9 */
/* Full (unmasked, non-causal) multi-head self-attention between the fused QKV
 * projection and the out-projection ("the
 * transformer's full self-attention ... a fused attention kernel (FlashAttention-
 * class)", L224).  The definition, per sequence b, head h, query i:
 *     s_j = scale * sum_d q_i[d] k_j[d];   p_j = exp(s_j - max_j s) / sum_j exp(s_j - max_j s);
 *     o_i[d] = sum_j p_j v_j[d]
 * Layout (R21): QKV [B*S, 3*H*Dh], row = token b*S + i, columns
 * [ q (H*Dh) | k (H*Dh) | v (H*Dh) ], head h at columns h*Dh .. h*Dh+Dh-1 of its
 * third; O [B*S, H*Dh].  fp64 throughout (subtracting the row maximum changes
 * nothing mathematically; it only keeps exp() in range). */
void oracle_attention(const float *QKV, int64_t B, int64_t S, int64_t H, int64_t Dh, double scale, double *O)
{
    const int64_t ld = 3 * H * Dh;
#pragma omp parallel for collapse(2) schedule(static)
    for (int64_t b = 0; b < B; ++b)
        for (int64_t h = 0; h < H; ++h) {
            double s[S];
            for (int64_t i = 0; i < S; ++i) {
                const float *q = QKV + (b * S + i) * ld + h * Dh;
                double mx = -INFINITY;
                for (int64_t j = 0; j < S; ++j) {
                    const float *k = QKV + (b * S + j) * ld + H * Dh + h * Dh;
                    double a = 0.0;
                    for (int64_t d = 0; d < Dh; ++d)
                        a += (double)q[d] * (double)k[d];
                    s[j] = scale * a;
                    if (s[j] > mx)
                        mx = s[j];
                }
                double l = 0.0;
                for (int64_t j = 0; j < S; ++j) {
                    s[j] = exp(s[j] - mx);
                    l += s[j];
                }
                for (int64_t d = 0; d < Dh; ++d) {
                    double a = 0.0;
                    for (int64_t j = 0; j < S; ++j)
                        a += s[j] * (double)QKV[(b * S + j) * ld + 2 * H * Dh + h * Dh + d];
                    O[(b * S + i) * H * Dh + h * Dh + d] = a / l;
                }
            }
        }
}

/* ------------------------------------------------------------ output cast */
/* One rounding of the fp64 result to the output dtype: dtype 0 = fp32 (C cast,
 * RNE), dtype 1 = bf16 (RNE, returned widened to fp32). */
void oracle_round_out(const double *y, int64_t n, int dtype, float *out)
{
    for (int64_t i = 0; i < n; ++i) {
        if (dtype == 0)
            out[i] = (float)y[i];
        else
            out[i] = oracle_bf16_bits_to_f32(oracle_f64_to_bf16_bits(y[i]));
    }
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
