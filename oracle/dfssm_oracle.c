/*
 * DF-SSM per-token decode step -- CPU ORACLE.  See dfssm_oracle.h for the contract.
 * TEST INFRASTRUCTURE ONLY: never linked, imported or called by the product path.
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fno-fast-math -fno-math-errno -fopenmp -shared -fPIC
 *
 * Parity pins (tests/test_oracle_*.py): every function below is pinned to a closed form,
 * an invariant, a brute-force sum or a dense float64 definition EXCEPT the end-to-end
 * numerical values of a whole model, which the paper gives no worked example for:
 *   whole-model values: parity unpinned (pinned only through its parts + batch/reset invariants).
 */
#include "dfssm_oracle.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------
 * Arithmetic mode (TEST-ONLY switch; the default, DFO_MODE_CONTRACT, is the oracle).
 *   DFO_MODE_CONTRACT  the arithmetic contract of DESIGN.md section 5.
 *   DFO_MODE_REVERSED  the same contract with every binary64 reduction summed in REVERSED index order:
 *                      the contract says the result does not depend on the summation tree;
 *                      tests/test_oracle_model.py checks that on the oracle itself, bit for bit.
 *   DFO_MODE_F64       diagnostic ("float64 everything"): every expression is evaluated in
 *                      binary64 with libm transcendentals and rounded once where the contract stores a binary32
 *                      value (activations, state).  A perfectly reasonable implementation -- and it departs from
 *                      the contract mode within a few steps because a quantiser input that differs in the last bit
 *                      eventually rounds the other way.  It exists to show why the contract is needed.
 * ------------------------------------------------------------------------------------------ */
static int g_mode = DFO_MODE_CONTRACT;
void dfo_set_mode(int mode) { g_mode = (mode == DFO_MODE_REVERSED || mode == DFO_MODE_F64) ? mode : DFO_MODE_CONTRACT; }
int dfo_get_mode(void) { return g_mode; }
/* index of the i-th term of a reduction over n terms */
static int red_idx(int i, int n) { return g_mode == DFO_MODE_REVERSED ? n - 1 - i : i; }

/* ------------------------------------------------------------------------------------------
 * Specified transcendentals.  Fixed sequences of binary32 operations.
 * ------------------------------------------------------------------------------------------ */

/* exp(x): clamp to [-87, 88] (below -87 -> 0); n = rint(x*log2(e)); Cody-Waite two-constant
 * reduction r = x - n*ln2 with fmaf; degree-7 Taylor polynomial in Horner form with the
 * coefficients 1/k! rounded to binary32; scale by 2^n through the exponent field. */
float dfo_sp_expf(float x)
{
    const float LOG2E  = 0x1.715476p+0f;      /* fl32(1/ln 2)               */
    const float LN2_HI = 0x1.63p-1f;          /* 0.693359375, 9 significant bits */
    const float LN2_LO = -0x1.bd0106p-13f;    /* fl32(ln 2 - LN2_HI)        */
    const float C2 = 0x1p-1f;                 /* 1/2!  */
    const float C3 = 0x1.555556p-3f;          /* 1/3!  */
    const float C4 = 0x1.555556p-5f;          /* 1/4!  */
    const float C5 = 0x1.111112p-7f;          /* 1/5!  */
    const float C6 = 0x1.6c16c2p-10f;         /* 1/6!  */
    const float C7 = 0x1.a01a02p-13f;         /* 1/7!  */
    if (x < -87.0f) return 0.0f;
    if (x > 88.0f) x = 88.0f;
    float n = rintf(x * LOG2E);
    float r = fmaf(n, -LN2_HI, x);
    r = fmaf(n, -LN2_LO, r);
    float p = C7;
    p = fmaf(p, r, C6);
    p = fmaf(p, r, C5);
    p = fmaf(p, r, C4);
    p = fmaf(p, r, C3);
    p = fmaf(p, r, C2);
    p = fmaf(p, r, 1.0f);
    p = fmaf(p, r, 1.0f);
    int32_t ni = (int32_t)n;                          /* in [-126, 127] */
    uint32_t bits = (uint32_t)(ni + 127) << 23;       /* 2^n, a normal number */
    float two_n;
    memcpy(&two_n, &bits, sizeof two_n);
    return p * two_n;
}

/* log(1+t) for t in [0,1]: s = t/(2+t); log1p(t) = 2*atanh(s) = 2*s*(1 + s^2/3 + ... + s^16/17) */
float dfo_sp_log1pf(float t)
{
    const float K1 = 0x1.555556p-2f;   /* 1/3  */
    const float K2 = 0x1.99999ap-3f;   /* 1/5  */
    const float K3 = 0x1.24924ap-3f;   /* 1/7  */
    const float K4 = 0x1.c71c72p-4f;   /* 1/9  */
    const float K5 = 0x1.745d18p-4f;   /* 1/11 */
    const float K6 = 0x1.3b13b2p-4f;   /* 1/13 */
    const float K7 = 0x1.111112p-4f;   /* 1/15 */
    const float K8 = 0x1.e1e1e2p-5f;   /* 1/17 */
    float s = t / (2.0f + t);
    float s2 = s * s;
    float p = K8;
    p = fmaf(p, s2, K7);
    p = fmaf(p, s2, K6);
    p = fmaf(p, s2, K5);
    p = fmaf(p, s2, K4);
    p = fmaf(p, s2, K3);
    p = fmaf(p, s2, K2);
    p = fmaf(p, s2, K1);
    p = fmaf(p, s2, 1.0f);
    return 2.0f * (s * p);
}

/* softplus(x) = max(x,0) + log1p(exp(-|x|)); returns x for x > 20 */
float dfo_sp_softplusf(float x)
{
    if (x > 20.0f) return x;
    float e = dfo_sp_expf(-fabsf(x));
    float l = dfo_sp_log1pf(e);
    float m = x > 0.0f ? x : 0.0f;
    return m + l;
}

float dfo_siluf(float x)
{
    return x / (1.0f + dfo_sp_expf(-x));
}

/* IEEE binary16 -> binary32, exact (subnormals kept) */
float dfo_half_to_float(uint16_t h)
{
    uint32_t sign = (uint32_t)(h >> 15) << 31;
    int32_t e = (h >> 10) & 0x1f;
    uint32_t m = h & 0x3ffu;
    float mag;
    if (e == 0) {
        mag = (float)m * 0x1p-24f;                    /* subnormal or zero: m * 2^-24 */
    } else if (e == 31) {
        uint32_t bits = 0x7f800000u | (m << 13);
        memcpy(&mag, &bits, 4);
    } else {
        uint32_t bits = ((uint32_t)(e - 15 + 127) << 23) | (m << 13);
        memcpy(&mag, &bits, 4);
    }
    uint32_t out;
    memcpy(&out, &mag, 4);
    out |= sign;
    memcpy(&mag, &out, 4);
    return mag;
}

/* ------------------------------------------------------------------------------------------
 * Step functions
 * ------------------------------------------------------------------------------------------ */

/* S0: int8 per-row embedding, "quantized to int8 per-row", tied with the head */
/* binary32 -> binary16, round to nearest even (IEEE 754 convertFormat: subnormals kept, overflow -> infinity, NaN stays NaN);
 * the inverse of dfo_half_to_float on every binary16 value.  Used by the fp16 state format (R24). */
uint16_t dfo_float_to_half(float f)
{
    uint32_t x;
    memcpy(&x, &f, 4);
    const uint32_t sign = (x >> 16) & 0x8000u;
    const uint32_t ax = x & 0x7fffffffu;
    if (ax >= 0x7f800000u) return (uint16_t)(sign | 0x7c00u | (ax > 0x7f800000u ? 0x200u : 0u));       /* inf / NaN */
    if (ax >= 0x477ff000u) return (uint16_t)(sign | 0x7c00u);          /* >= 65520 rounds to infinity */
    if (ax < 0x33000001u) return (uint16_t)sign;                        /* <= 2^-25: rounds to zero (2^-25 itself ties to even = 0) */
    int e = (int)(ax >> 23) - 127;                                      /* unbiased exponent */
    uint32_t m = (ax & 0x7fffffu) | 0x800000u;                          /* 24-bit significand */
    int shift;                                                          /* bits dropped from the significand */
    uint32_t he;
    if (e < -14) { shift = 13 + (-14 - e); he = 0; }                    /* binary16 subnormal */
    else { shift = 13; he = (uint32_t)(e + 15); }
    uint32_t q = m >> shift;
    const uint32_t rem = m & ((1u << shift) - 1u), half = 1u << (shift - 1);
    if (rem > half || (rem == half && (q & 1u))) ++q;                   /* ties to even; a carry walks into the exponent */
    uint32_t h = he == 0 ? q : ((he << 10) + (q - 0x400u));
    return (uint16_t)(sign | h);
}

/* the fp16 state format (R24): every state value is replaced by float(half(value)) after the step's update and
 * readout (the readout of the step itself used the unrounded binary32 values) */
void dfo_round_state_f16(float* H, size_t n)
{
    for (size_t i = 0; i < n; ++i) H[i] = dfo_half_to_float(dfo_float_to_half(H[i]));
}

static float silu_mode(float x)
{
    if (g_mode == DFO_MODE_F64) return (float)((double)x / (1.0 + exp(-(double)x)));
    return dfo_siluf(x);
}

void dfo_embed(const int8_t* E_row, float e_s, int d, float* u)
{
    for (int k = 0; k < d; ++k) u[k] = e_s * (float)E_row[k];
}

/* S1/S6/S8: RMSNorm (P:407-408 list the norms) + per-token absmax int8 quantiser (paper silent;
 * DESIGN.md R4).  The positive scalar rstd cancels in x*127/max|x|, so the int8 codes are taken
 * from t = v*w and rstd is folded into the scale (R13). */
void dfo_norm_quant(const float* v, const float* w, int d, float eps,
                    int8_t* q, float* s, float* rstd_out, float* amax_out)
{
    double ss = 0.0;
    for (int i = 0; i < d; ++i) { const int k = red_idx(i, d); ss += (double)v[k] * (double)v[k]; }
    float ms = (float)(ss / (double)d);
    float rstd = 1.0f / sqrtf(ms + eps);
    if (g_mode == DFO_MODE_F64) rstd = (float)(1.0 / sqrt(ss / (double)d + (double)eps));
    float amax = 0.0f;
    for (int k = 0; k < d; ++k) {
        float a = fabsf(v[k] * w[k]);
        if (a > amax) amax = a;
    }
    if (amax == 0.0f) {
        for (int k = 0; k < d; ++k) q[k] = 0;
        *s = 0.0f;
    } else {
        float inv = 127.0f / amax;
        for (int k = 0; k < d; ++k) {
            float f = rintf((v[k] * w[k]) * inv);     /* ties to even */
            if (g_mode == DFO_MODE_F64) f = (float)rint((double)v[k] * (double)w[k] * (127.0 / (double)amax));
            if (f > 127.0f) f = 127.0f;
            if (f < -127.0f) f = -127.0f;
            q[k] = (int8_t)f;
        }
        *s = (amax * rstd) / 127.0f;
        if (g_mode == DFO_MODE_F64) *s = (float)((double)amax * (1.0 / sqrt(ss / (double)d + (double)eps)) / 127.0);
    }
    if (rstd_out) *rstd_out = rstd;
    if (amax_out) *amax_out = amax;
}

/* S2/S7: bit 1 -> +1, bit 0 -> -1; element k = 32*word + bit */
void dfo_sign_matvec(const uint32_t* sign, int rows, int K, const int8_t* xq, int32_t* acc)
{
    const int W = K / 32;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < rows; ++i) {
        int32_t a = 0;
        for (int w = 0; w < W; ++w) {
            uint32_t bits = sign[(size_t)i * W + w];
            for (int b = 0; b < 32; ++b) {
                int32_t x = xq[32 * w + b];
                a += ((bits >> b) & 1u) ? x : -x;
            }
        }
        acc[i] = a;
    }
}

/* S3 stage 1: LoRA down-projection W_B x of Eq. 3 on the int8 activations (R7) */
void dfo_lora_down(const int8_t* A, int r, int K, const int8_t* xq, int32_t* t)
{
    for (int j = 0; j < r; ++j) {
        int32_t a = 0;
        for (int k = 0; k < K; ++k) a += (int32_t)A[(size_t)j * K + k] * (int32_t)xq[k];
        t[j] = a;
    }
}

/* Format variant (R25): the 17-level scaffold of Eq. 1 / Eq. 3,
 * W_scaffold in {-1, -14/16, ..., 14/16, 1} = level / 8 with level = m - 8, m in [0, 16] stored as five bit planes:
 * bit b of lvl[i][w][p] is bit p of m of element k = 32*w + b.  acc_i = sum_k level_ik * q_k, exact int32
 * (the row scale of the blob multiplies this integer sum, i.e. it holds the paper's scale / 8). */
void dfo_level_matvec(const uint32_t* lvl, int rows, int K, const int8_t* xq, int32_t* acc)
{
    const int W = K / 32;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < rows; ++i) {
        int32_t a = 0;
        for (int w = 0; w < W; ++w) {
            const uint32_t* pl = lvl + ((size_t)i * W + w) * 5;
            for (int b = 0; b < 32; ++b) {
                int m = 0;
                for (int p = 0; p < 5; ++p) m |= (int)((pl[p] >> b) & 1u) << p;
                a += (int32_t)(m - 8) * (int32_t)xq[32 * w + b];
            }
        }
        acc[i] = a;
    }
}

/* Format variant: int4 LoRA (Table 4).  Element 2i of a row is the low nibble of byte i, element 2i + 1 the high
 * nibble; a nibble is a two's-complement 4-bit integer in [-8, 7].  n = values per row (even). */
void dfo_unpack_int4(const uint8_t* packed, int rows, int n, int8_t* out)
{
    for (int i = 0; i < rows; ++i)
        for (int j = 0; j < n; ++j) {
            const int nib = (packed[(size_t)i * (n / 2) + j / 2] >> (4 * (j & 1))) & 0xF;
            out[(size_t)i * n + j] = (int8_t)(nib >= 8 ? nib - 16 : nib);
        }
}

/* S3 stage 2 + dequantisation: y = W_scaffold x + W_A (W_B x), Eq. 3, alpha folded in scales */
void dfo_proj_epilogue(const int32_t* acc, const int32_t* t, const uint16_t* row_scale_f16,
                       const float* a_s, const int8_t* B, const float* b_s,
                       int rows, int r, float s_x, float* out)
{
    float* v = (float*)malloc(sizeof(float) * (size_t)r);
    for (int j = 0; j < r; ++j) v[j] = a_s[j] * (float)t[j];
    for (int i = 0; i < rows; ++i) {
        double lo = 0.0;
        for (int jj = 0; jj < r; ++jj) { const int j = red_idx(jj, r); lo += (double)(float)B[(size_t)i * r + j] * (double)v[j]; }
        float lo_f = (float)lo;
        float m1 = dfo_half_to_float(row_scale_f16[i]) * (float)acc[i];
        float m2 = b_s[i] * lo_f;
        out[i] = s_x * (m1 + m2);
        if (g_mode == DFO_MODE_F64) {
            double lod = 0.0;
            for (int j = 0; j < r; ++j) lod += (double)B[(size_t)i * r + j] * ((double)a_s[j] * (double)t[j]);
            out[i] = (float)((double)s_x * ((double)dfo_half_to_float(row_scale_f16[i]) * (double)acc[i] + (double)b_s[i] * lod));
        }
    }
    free(v);
}

/* S4: "convolution step (stateful shift register)"; SiLU after the conv (R9) */
void dfo_conv_step(float* state, const float* w, const float* bias, const float* xin, int C,
                   float* out)
{
    for (int c = 0; c < C; ++c) {
        float s0 = state[3 * c + 0], s1 = state[3 * c + 1], s2 = state[3 * c + 2];
        float xn = xin[c];
        float o = bias[c];
        o = fmaf(w[4 * c + 0], s0, o);
        o = fmaf(w[4 * c + 1], s1, o);
        o = fmaf(w[4 * c + 2], s2, o);
        o = fmaf(w[4 * c + 3], xn, o);
        state[3 * c + 0] = s1;
        state[3 * c + 1] = s2;
        state[3 * c + 2] = xn;
        if (g_mode == DFO_MODE_F64)
            o = (float)((double)bias[c] + (double)w[4 * c + 0] * s0 + (double)w[4 * c + 1] * s1 + (double)w[4 * c + 2] * s2 + (double)w[4 * c + 3] * xn);
        out[c] = silu_mode(o);
    }
}

/* S5: h = A h + (x*dt) (x) B  (Table 12, "Correct" column); y = C.h + D x on the UPDATED
 * state (R11); head h reads B/C group h / (nheads/ngroups) (R12) */
void dfo_ssm_step(float* H, const float* x, const float* Bv, const float* Cv, const float* dt,
                  const float* A, const float* D, int nheads, int headdim, int d_state,
                  int ngroups, float* y)
{
    const int hpg = nheads / ngroups;
#pragma omp parallel for schedule(static)
    for (int h = 0; h < nheads; ++h) {
        const float dA = g_mode == DFO_MODE_F64 ? (float)exp((double)dt[h] * (double)A[h]) : dfo_sp_expf(dt[h] * A[h]);
        const float* Bg = Bv + (size_t)(h / hpg) * d_state;
        const float* Cg = Cv + (size_t)(h / hpg) * d_state;
        for (int p = 0; p < headdim; ++p) {
            const float xv = x[h * headdim + p];
            const float dtx = dt[h] * xv;
            float* Hr = H + ((size_t)h * headdim + p) * d_state;
            double a = 0.0;
            if (g_mode == DFO_MODE_REVERSED) a += (double)D[h] * (double)xv;      /* the last term first */
            for (int i = 0; i < d_state; ++i) {
                const int n = red_idx(i, d_state);
                float hn = fmaf(dA, Hr[n], dtx * Bg[n]);
                if (g_mode == DFO_MODE_F64) hn = (float)((double)dA * (double)Hr[n] + (double)dt[h] * (double)xv * (double)Bg[n]);
                Hr[n] = hn;
                a += (double)Cg[n] * (double)hn;
            }
            if (g_mode != DFO_MODE_REVERSED) a += (double)D[h] * (double)xv;
            y[h * headdim + p] = (float)a;
        }
    }
}

/* S6: norm(y * silu(z)) -- gate first */
void dfo_gate(const float* y, const float* z, int n, float* g)
{
    for (int i = 0; i < n; ++i) g[i] = g_mode == DFO_MODE_F64 ? (float)((double)y[i] * ((double)z[i] / (1.0 + exp(-(double)z[i])))) : y[i] * dfo_siluf(z[i]);
}

/* S8: tied int8 LM head on the quantised final hidden (R16) */
void dfo_lm_head(const int8_t* E, const float* e_s, int vocab, int d, const int8_t* hq, float s_h,
                 int32_t* acc_or_null, float* logits)
{
#pragma omp parallel for schedule(static)
    for (int v = 0; v < vocab; ++v) {
        int32_t a = 0;
        const int8_t* row = E + (size_t)v * d;
        for (int k = 0; k < d; ++k) a += (int32_t)row[k] * (int32_t)hq[k];
        if (acc_or_null) acc_or_null[v] = a;
        logits[v] = (float)a * (s_h * e_s[v]);
    }
}

/* Temperature / top-k sampling of one token from a logits vector (the generation loop the paper implies; the paper gives no
 * sampler: DESIGN.md R23).  Greedy decode is the case top_k == 1 (or temperature <= 0).
 *   1. the top_k largest logits, equal logits ordered by LOWER index first: ranks 0 .. k-1;
 *   2. w_r = sp_expf((l_r - l_0) / temperature)        (binary32 operations, the specified exp);
 *   3. c_r = w_0 + ... + w_r accumulated in binary64 in rank order;
 *   4. the smallest rank r with c_r > (double)u * c_{k-1} (u in [0,1) is the caller's uniform random number; r = k-1 if none).
 * Returns the vocabulary index of that rank.  O(k * n): a plain selection, no sort. */
int dfo_sample(const float* logits, int n, float temperature, int top_k, float u)
{
    if (top_k < 1) top_k = 1;
    if (top_k > n) top_k = n;
    if (top_k > 64) top_k = 64;
    if (!(temperature > 0.0f)) top_k = 1;
    int idx[64];
    float val[64];
    int prev_i = -1;
    float prev_v = 0.0f;
    for (int r = 0; r < top_k; ++r) {
        int bi = -1;
        float bv = 0.0f;
        for (int i = 0; i < n; ++i) {
            const float x = logits[i];
            /* candidates strictly after the previous pick in the order (value descending, index ascending) */
            if (r > 0 && !(x < prev_v || (x == prev_v && i > prev_i))) continue;
            if (bi < 0 || x > bv) { bi = i; bv = x; }       /* the first (lowest) index wins among equals */
        }
        idx[r] = bi; val[r] = bv;
        prev_i = bi; prev_v = bv;
    }
    if (top_k == 1) return idx[0];
    double c[64];
    double run = 0.0;
    for (int r = 0; r < top_k; ++r) {
        const float w = dfo_sp_expf((val[r] - val[0]) / temperature);
        run += (double)w;
        c[r] = run;
    }
    const double thr = (double)u * run;
    for (int r = 0; r < top_k; ++r)
        if (c[r] > thr) return idx[r];
    return idx[top_k - 1];
}

int dfo_argmax(const float* logits, int n)
{
    int best = 0;
    for (int i = 1; i < n; ++i)
        if (logits[i] > logits[best]) best = i;
    return best;
}

/* ------------------------------------------------------------------------------------------
 * Whole model: blob parsing + the step
 * ------------------------------------------------------------------------------------------ */

typedef struct {
    const float* norm_w;
    const uint32_t* in_sign; const uint16_t* in_row_scale;
    const int8_t* in_A; const float* in_a_s; const int8_t* in_B; const float* in_b_s;
    const float* conv_w; const float* conv_b;
    const float* A_log; const float* dt_bias; const float* D;
    const float* gnorm_w;
    const uint32_t* out_sign; const uint16_t* out_row_scale;
    const int8_t* out_A; const float* out_a_s; const int8_t* out_B; const float* out_b_s;
    int8_t* own[4];            /* int4 LoRA: the unpacked copies of A / B (in, out) this layer owns */
} dfo_layer;

struct dfo_model {
    uint8_t* blob;
    int n_layers, d_model, d_inner, headdim, d_state, ngroups, d_conv, vocab, r;
    int nheads, d_in_proj, conv_dim;
    int fmt;                    /* blob header word 52: bit 0 = 17-level scaffold, bit 1 = int4 LoRA (R25) */
    float eps;
    int max_batch, last_batch;
    dfo_layer* layers;
    const int8_t* emb; const float* emb_s; const float* normf_w;
    float* ssm;    /* [layer][seq][nheads*headdim*d_state] */
    float* conv;   /* [layer][seq][conv_dim*3] */
    float* logits; /* [seq][vocab] */
    int32_t* next; /* [seq] */
    float* hidden; /* [seq][d_model] */
    int taps_on;
    int state_fp16;             /* DESIGN.md R24: the SSM state is stored as binary16 between steps */
    uint8_t* taps; /* [layer][seq][tap_stride] */
    size_t tap_off[DFO_TAP_COUNT + 1];
};

static size_t align64(size_t x) { return (x + 63) & ~(size_t)63; }

static int32_t rd_i32(const uint8_t* p) { int32_t v; memcpy(&v, p, 4); return v; }

dfo_model* dfo_load(const void* blob, size_t nbytes, int max_batch, char* err, size_t errlen)
{
#define FAIL(msg) do { if (err && errlen) snprintf(err, errlen, "%s", msg); dfo_free(m); return NULL; } while (0)
    dfo_model* m = (dfo_model*)calloc(1, sizeof *m);
    const uint8_t* b = (const uint8_t*)blob;
    if (!m) return NULL;
    if (nbytes < 256 || memcmp(b, "DFSSMW1\0", 8) != 0) FAIL("bad magic or short blob");
    if (rd_i32(b + 8) != 1) FAIL("unsupported blob version");
    m->n_layers = rd_i32(b + 12); m->d_model = rd_i32(b + 16); m->d_inner = rd_i32(b + 20);
    m->headdim = rd_i32(b + 24);  m->d_state = rd_i32(b + 28); m->ngroups = rd_i32(b + 32);
    m->d_conv = rd_i32(b + 36);   m->vocab = rd_i32(b + 40);   m->r = rd_i32(b + 44);
    memcpy(&m->eps, b + 48, 4);
    m->fmt = rd_i32(b + 52);
    if (m->fmt < 0 || m->fmt > 3) FAIL("unknown weight format");
    if ((m->fmt & 2) && (m->r % 2)) FAIL("int4 LoRA needs an even rank");
    uint64_t total; memcpy(&total, b + 56, 8);
    if (total != (uint64_t)nbytes) FAIL("blob size does not match header");
    if (m->d_conv != 4) FAIL("d_conv must be 4");
    if (m->n_layers < 0 || m->d_model <= 0 || m->d_model % 32 || m->d_inner <= 0 || m->d_inner % 32 ||
        m->headdim <= 0 || m->d_inner % m->headdim || m->ngroups <= 0 || m->d_state <= 0 ||
        m->vocab <= 0 || m->r <= 0 || max_batch < 1)
        FAIL("bad shape");
    m->nheads = m->d_inner / m->headdim;
    if (m->nheads % m->ngroups) FAIL("nheads not divisible by ngroups");
    m->d_in_proj = 2 * m->d_inner + 2 * m->ngroups * m->d_state + m->nheads;
    m->conv_dim = m->d_inner + 2 * m->ngroups * m->d_state;
    m->max_batch = max_batch;

    /* walk the canonical tensor order */
    size_t off = 256;
#define TAKE(ptr, type, count) do { off = align64(off); (ptr) = (const type*)(m->blob + off); \
                                    off += sizeof(type) * (size_t)(count); } while (0)
    m->blob = (uint8_t*)malloc(nbytes);
    if (!m->blob) FAIL("out of memory");
    memcpy(m->blob, blob, nbytes);
    m->layers = (dfo_layer*)calloc((size_t)(m->n_layers > 0 ? m->n_layers : 1), sizeof(dfo_layer));
    const size_t dm = m->d_model, di = m->d_inner, dip = m->d_in_proj, r = m->r;
    for (int l = 0; l < m->n_layers; ++l) {
        dfo_layer* L = &m->layers[l];
        TAKE(L->norm_w, float, dm);
        const size_t planes = (m->fmt & 1) ? 5 : 1;      /* in_sign / out_sign point at the bit planes then */
        const int i4 = (m->fmt & 2) != 0;
#define TAKE_LORA(dst, slot, rows_, n_) do { \
            if (i4) { const uint8_t* pk; TAKE(pk, uint8_t, (size_t)(rows_) * (n_) / 2); \
                      L->own[slot] = (int8_t*)malloc((size_t)(rows_) * (n_)); if (!L->own[slot]) FAIL("out of memory"); \
                      dfo_unpack_int4(pk, (int)(rows_), (int)(n_), L->own[slot]); (dst) = L->own[slot]; } \
            else TAKE(dst, int8_t, (size_t)(rows_) * (n_)); } while (0)
        TAKE(L->in_sign, uint32_t, dip * (dm / 32) * planes);
        TAKE(L->in_row_scale, uint16_t, dip);
        TAKE_LORA(L->in_A, 0, r, dm);
        TAKE(L->in_a_s, float, r);
        TAKE_LORA(L->in_B, 1, dip, r);
        TAKE(L->in_b_s, float, dip);
        TAKE(L->conv_w, float, (size_t)m->conv_dim * 4);
        TAKE(L->conv_b, float, m->conv_dim);
        TAKE(L->A_log, float, m->nheads);
        TAKE(L->dt_bias, float, m->nheads);
        TAKE(L->D, float, m->nheads);
        TAKE(L->gnorm_w, float, di);
        TAKE(L->out_sign, uint32_t, dm * (di / 32) * planes);
        TAKE(L->out_row_scale, uint16_t, dm);
        TAKE_LORA(L->out_A, 2, r, di);
        TAKE(L->out_a_s, float, r);
        TAKE_LORA(L->out_B, 3, dm, r);
        TAKE(L->out_b_s, float, dm);
    }
    TAKE(m->emb, int8_t, (size_t)m->vocab * dm);
    TAKE(m->emb_s, float, m->vocab);
    TAKE(m->normf_w, float, dm);
    if (align64(off) != nbytes) FAIL("blob size does not match the shape");

    size_t ssm_n = (size_t)m->nheads * m->headdim * m->d_state;
    size_t nl = (size_t)(m->n_layers > 0 ? m->n_layers : 1);
    m->ssm = (float*)calloc(nl * max_batch * ssm_n, sizeof(float));
    m->conv = (float*)calloc(nl * max_batch * (size_t)m->conv_dim * 3, sizeof(float));
    m->logits = (float*)calloc((size_t)max_batch * m->vocab, sizeof(float));
    m->next = (int32_t*)calloc((size_t)max_batch, sizeof(int32_t));
    m->hidden = (float*)calloc((size_t)max_batch * dm, sizeof(float));
    if (!m->ssm || !m->conv || !m->logits || !m->next || !m->hidden) FAIL("out of memory");

    size_t sizes[DFO_TAP_COUNT] = {
        dm, 4, 4 * dip, 4 * r, 4 * dip, 4 * (size_t)m->conv_dim, 4 * (size_t)m->nheads,
        4 * di, 4 * di, di, 4, 4 * dm, 4 * r, 4 * dm };
    size_t o = 0;
    for (int i = 0; i < DFO_TAP_COUNT; ++i) { m->tap_off[i] = o; o = align64(o + sizes[i]); }
    m->tap_off[DFO_TAP_COUNT] = o;
    return m;
#undef TAKE
#undef FAIL
}

void dfo_free(dfo_model* m)
{
    if (!m) return;
    if (m->layers)
        for (int l = 0; l < m->n_layers; ++l)
            for (int k = 0; k < 4; ++k) free(m->layers[l].own[k]);
    free(m->blob); free(m->layers); free(m->ssm); free(m->conv); free(m->logits);
    free(m->next); free(m->hidden); free(m->taps); free(m);
}

void dfo_set_threads(int n)
{
#ifdef _OPENMP
    if (n <= 0) n = omp_get_num_procs();
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int dfo_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void dfo_set_state_fp16(dfo_model* m, int on) { m->state_fp16 = on ? 1 : 0; }

void dfo_enable_taps(dfo_model* m, int on)
{
    m->taps_on = on;
    if (on && !m->taps) {
        size_t nl = (size_t)(m->n_layers > 0 ? m->n_layers : 1);
        m->taps = (uint8_t*)calloc(nl * m->max_batch * m->tap_off[DFO_TAP_COUNT], 1);
    }
}

static size_t ssm_elems(const dfo_model* m) { return (size_t)m->nheads * m->headdim * m->d_state; }

float* dfo_ssm_state(dfo_model* m, int layer, int seq)
{
    return m->ssm + ((size_t)layer * m->max_batch + seq) * ssm_elems(m);
}

float* dfo_conv_state(dfo_model* m, int layer, int seq)
{
    return m->conv + ((size_t)layer * m->max_batch + seq) * (size_t)m->conv_dim * 3;
}

/* "State tensors for SSM and convolution are preallocated and persist across tokens";
 * reset zeroes them */
void dfo_reset(dfo_model* m, int seq)
{
    for (int l = 0; l < m->n_layers; ++l)
        for (int s = 0; s < m->max_batch; ++s) {
            if (seq >= 0 && s != seq) continue;
            memset(dfo_ssm_state(m, l, s), 0, ssm_elems(m) * sizeof(float));
            memset(dfo_conv_state(m, l, s), 0, (size_t)m->conv_dim * 3 * sizeof(float));
        }
}

static uint8_t* tap_ptr(const dfo_model* m, int layer, int which, int seq)
{
    return m->taps + ((size_t)layer * m->max_batch + seq) * m->tap_off[DFO_TAP_COUNT] + m->tap_off[which];
}

const void* dfo_tap(const dfo_model* m, int layer, int which, int seq, size_t* nbytes)
{
    if (!m->taps || layer < 0 || layer >= m->n_layers || which < 0 || which >= DFO_TAP_COUNT ||
        seq < 0 || seq >= m->max_batch)
        return NULL;
    if (nbytes) *nbytes = m->tap_off[which + 1] - m->tap_off[which];   /* padded size */
    return tap_ptr(m, layer, which, seq);
}

#define TAP(which, src, bytes) do { if (m->taps_on) memcpy(tap_ptr(m, l, which, s), (src), (bytes)); } while (0)

/* one sequence, one token: S0, L x (S1..S7), S8 */
static void step_one(dfo_model* m, int s, int32_t tok)
{
    const int dm = m->d_model, di = m->d_inner, dip = m->d_in_proj, r = m->r;
    const int gs = m->ngroups * m->d_state;
    float* u = m->hidden + (size_t)s * dm;
    int8_t* xq = (int8_t*)malloc((size_t)(dm > di ? dm : di));
    int32_t* acc = (int32_t*)malloc(sizeof(int32_t) * (size_t)(dip > dm ? dip : dm));
    int32_t* t = (int32_t*)malloc(sizeof(int32_t) * (size_t)r);
    float* zx = (float*)malloc(sizeof(float) * (size_t)dip);
    float* xbc = (float*)malloc(sizeof(float) * (size_t)m->conv_dim);
    float* dt = (float*)malloc(sizeof(float) * (size_t)m->nheads);
    float* An = (float*)malloc(sizeof(float) * (size_t)m->nheads);
    float* y = (float*)malloc(sizeof(float) * (size_t)di);
    float* g = (float*)malloc(sizeof(float) * (size_t)di);
    float* o = (float*)malloc(sizeof(float) * (size_t)dm);
    float sx;

    dfo_embed(m->emb + (size_t)tok * dm, m->emb_s[tok], dm, u);                          /* S0 */
    for (int l = 0; l < m->n_layers; ++l) {
        const dfo_layer* L = &m->layers[l];
        dfo_norm_quant(u, L->norm_w, dm, m->eps, xq, &sx, NULL, NULL);                   /* S1 */
        TAP(DFO_TAP_XQ_IN, xq, (size_t)dm); TAP(DFO_TAP_S_IN, &sx, 4);
        if (m->fmt & 1) dfo_level_matvec(L->in_sign, dip, dm, xq, acc);                  /* S2, 17-level variant */
        else dfo_sign_matvec(L->in_sign, dip, dm, xq, acc);                              /* S2 */
        dfo_lora_down(L->in_A, r, dm, xq, t);                                            /* S3 */
        dfo_proj_epilogue(acc, t, L->in_row_scale, L->in_a_s, L->in_B, L->in_b_s, dip, r, sx, zx);
        TAP(DFO_TAP_ACC_IN, acc, 4 * (size_t)dip); TAP(DFO_TAP_T_IN, t, 4 * (size_t)r);
        TAP(DFO_TAP_ZXBCDT, zx, 4 * (size_t)dip);
        /* split z | x | B | C | dt  (R8) */
        const float* z = zx;
        const float* xBC_raw = zx + di;
        const float* dt_raw = zx + di + m->conv_dim;
        dfo_conv_step(dfo_conv_state(m, l, s), L->conv_w, L->conv_b, xBC_raw, m->conv_dim, xbc);  /* S4 */
        TAP(DFO_TAP_XBC_CONV, xbc, 4 * (size_t)m->conv_dim);
        for (int h = 0; h < m->nheads; ++h) {                                            /* S5 */
            dt[h] = dfo_sp_softplusf(dt_raw[h] + L->dt_bias[h]);
            An[h] = -dfo_sp_expf(L->A_log[h]);
            if (g_mode == DFO_MODE_F64) {
                const double xx = (double)dt_raw[h] + (double)L->dt_bias[h];
                dt[h] = (float)(xx > 20.0 ? xx : log1p(exp(xx)));
                An[h] = (float)(-exp((double)L->A_log[h]));
            }
        }
        TAP(DFO_TAP_DT, dt, 4 * (size_t)m->nheads);
        dfo_ssm_step(dfo_ssm_state(m, l, s), xbc, xbc + di, xbc + di + gs, dt, An, L->D,
                     m->nheads, m->headdim, m->d_state, m->ngroups, y);
        if (m->state_fp16) dfo_round_state_f16(dfo_ssm_state(m, l, s), ssm_elems(m));
        TAP(DFO_TAP_Y, y, 4 * (size_t)di);
        dfo_gate(y, z, di, g);                                                           /* S6 */
        TAP(DFO_TAP_G, g, 4 * (size_t)di);
        dfo_norm_quant(g, L->gnorm_w, di, m->eps, xq, &sx, NULL, NULL);
        TAP(DFO_TAP_GQ, xq, (size_t)di); TAP(DFO_TAP_S_G, &sx, 4);
        if (m->fmt & 1) dfo_level_matvec(L->out_sign, dm, di, xq, acc);                  /* S7, 17-level variant */
        else dfo_sign_matvec(L->out_sign, dm, di, xq, acc);                              /* S7 */
        dfo_lora_down(L->out_A, r, di, xq, t);
        dfo_proj_epilogue(acc, t, L->out_row_scale, L->out_a_s, L->out_B, L->out_b_s, dm, r, sx, o);
        TAP(DFO_TAP_ACC_OUT, acc, 4 * (size_t)dm); TAP(DFO_TAP_T_OUT, t, 4 * (size_t)r);
        for (int k = 0; k < dm; ++k) u[k] = u[k] + o[k];                                 /* residual */
        TAP(DFO_TAP_HIDDEN, u, 4 * (size_t)dm);
    }
    dfo_norm_quant(u, m->normf_w, dm, m->eps, xq, &sx, NULL, NULL);                      /* S8 */
    float* lg = m->logits + (size_t)s * m->vocab;
    dfo_lm_head(m->emb, m->emb_s, m->vocab, dm, xq, sx, NULL, lg);
    m->next[s] = dfo_argmax(lg, m->vocab);

    free(xq); free(acc); free(t); free(zx); free(xbc); free(dt); free(An); free(y); free(g); free(o);
}

/* sequences are independent: own conv + SSM state, no cross-sequence term */
int dfo_step(dfo_model* m, const int32_t* tokens, int batch)
{
    if (!m || !tokens || batch < 1 || batch > m->max_batch) return -1;
    for (int s = 0; s < batch; ++s)
        if (tokens[s] < 0 || tokens[s] >= m->vocab) return -2;
    for (int s = 0; s < batch; ++s) step_one(m, s, tokens[s]);
    m->last_batch = batch;
    return 0;
}

const float* dfo_logits(const dfo_model* m) { return m->logits; }
const int32_t* dfo_next_tokens(const dfo_model* m) { return m->next; }
const float* dfo_hidden(const dfo_model* m) { return m->hidden; }

int dfo_shape(const dfo_model* m, int32_t out[12])
{
    int32_t v[12] = { m->n_layers, m->d_model, m->d_inner, m->headdim, m->d_state, m->ngroups,
                      m->d_conv, m->vocab, m->r, m->nheads, m->d_in_proj, m->conv_dim };
    memcpy(out, v, sizeof v);
    return 0;
}
