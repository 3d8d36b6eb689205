/*
 * DF-SSM per-token decode step -- CPU ORACLE (test infrastructure, NOT a product path).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this.  It shares no code with paper_2606_10932_b200/ (the CUDA path).
 *
 * Plain C99, one translation unit, no intrinsics.  Every function restates one passage
 * of /root/reference/PAPER.md ("P:NN" = line NN) or one reading listed in DESIGN.md §4.
 * Arithmetic contract: integer parts exact int32; each elementwise float
 * op is ONE IEEE binary32 operation in the order written here (compile with
 * -ffp-contract=off; fused ops are spelled fmaf); every floating reduction is accumulated
 * in binary64 from exact binary32 x binary32 products and rounded to binary32 once;
 * exp / log1p / softplus are the fixed op sequences dfo_sp_* below, never libm.
 */
#ifndef DFSSM_ORACLE_H
#define DFSSM_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---------- specified transcendentals ---------- */
float dfo_sp_expf(float x);
float dfo_sp_log1pf(float t);      /* t in [0, 1] */
float dfo_sp_softplusf(float x);
float dfo_siluf(float x);          /* x / (1 + exp(-x)) */
float dfo_half_to_float(uint16_t h);

/* ---------- step functions, one per row of SURVEY §8(a) ---------- */

/* S0  u[k] = e_s * float(E_row[k]) */
void dfo_embed(const int8_t* E_row, float e_s, int d, float* u);

/* S1/S6/S8  RMSNorm fused with the per-token absmax int8 quantiser (R4, R13):
 *   rstd = 1/sqrt(mean(v^2)+eps);  t_k = v_k*w_k;  amax = max|t_k|;
 *   q_k = clamp(rint(t_k * (127/amax)), +-127);  s = (amax*rstd)/127   (amax==0 -> q=0, s=0)
 * so that s*q_k ~= v_k*rstd*w_k. */
void dfo_norm_quant(const float* v, const float* w, int d, float eps,
                    int8_t* q, float* s, float* rstd, float* amax);

/* S2/S7  acc_i = sum_k sign_ik * xq_k, sign in {-1,+1}, exact int32 */
void dfo_sign_matvec(const uint32_t* sign, int rows, int K, const int8_t* xq, int32_t* acc);

/* S3 stage 1  t_j = sum_k A_jk * xq_k, exact int32                    (Eq. 3) */
void dfo_lora_down(const int8_t* A, int r, int K, const int8_t* xq, int32_t* t);
/* format variants (R25): 17-level scaffold as five bit planes [rows][K/32][5]; int4 pairs per byte */
void dfo_level_matvec(const uint32_t* lvl, int rows, int K, const int8_t* xq, int32_t* acc);
void dfo_unpack_int4(const uint8_t* packed, int rows, int n, int8_t* out);

/* S3 stage 2 + epilogue  out_i = s_x*( w_s[i]*float(acc_i) + b_s[i]*lo_i ),
 *   lo_i = round32( sum_j float(B_ij) * (a_s[j]*float(t_j)) )        (Eq. 3) */
void dfo_proj_epilogue(const int32_t* acc, const int32_t* t, const uint16_t* row_scale_f16,
                       const float* a_s, const int8_t* B, const float* b_s,
                       int rows, int r, float s_x, float* out);

/* S4  causal depthwise 4-tap conv step + SiLU over C channels; state [C][3] oldest first,
 *     w [C][4] with tap 3 on the newest sample */
void dfo_conv_step(float* state, const float* w, const float* bias, const float* xin, int C,
                   float* out);

/* S5  H <- dA*H + (dt*x) (x) B ; y = C.H + D*x, with dA_h = exp(dt_h*A_h); dt is the
 *     POST-softplus step size, A_h = -exp(A_log_h) (negative)         (Table 12) */
void dfo_ssm_step(float* H, const float* x, const float* Bv, const float* Cv, const float* dt,
                  const float* A, const float* D, int nheads, int headdim, int d_state,
                  int ngroups, float* y);

/* S6 (first half)  g = y * silu(z)   -- gate first, then norm */
void dfo_gate(const float* y, const float* z, int n, float* g);

/* S8  acc_v = sum_k E_vk*hq_k (int32); logit_v = float(acc_v) * (s_h*e_s[v]) */
void dfo_lm_head(const int8_t* E, const float* e_s, int vocab, int d, const int8_t* hq, float s_h,
                 int32_t* acc_or_null, float* logits);
int dfo_argmax(const float* logits, int n);   /* lowest index on ties */

/* ---------- whole model ---------- */
typedef struct dfo_model dfo_model;

/* taps (`which` of dfo_tap): per layer, per sequence */
enum {
    DFO_TAP_XQ_IN = 0,   /* int8  [d_model]   */
    DFO_TAP_S_IN,        /* f32   [1]         */
    DFO_TAP_ACC_IN,      /* int32 [d_in_proj] */
    DFO_TAP_T_IN,        /* int32 [r]         */
    DFO_TAP_ZXBCDT,      /* f32   [d_in_proj] */
    DFO_TAP_XBC_CONV,    /* f32   [conv_dim]  post conv+silu */
    DFO_TAP_DT,          /* f32   [nheads]    post softplus */
    DFO_TAP_Y,           /* f32   [d_inner]   */
    DFO_TAP_G,           /* f32   [d_inner]   y*silu(z) */
    DFO_TAP_GQ,          /* int8  [d_inner]   */
    DFO_TAP_S_G,         /* f32   [1]         */
    DFO_TAP_ACC_OUT,     /* int32 [d_model]   */
    DFO_TAP_T_OUT,       /* int32 [r]         */
    DFO_TAP_HIDDEN,      /* f32   [d_model]   residual stream after the layer */
    DFO_TAP_COUNT
};

/* blob is copied; returns NULL and fills err on a malformed blob */
dfo_model* dfo_load(const void* blob, size_t nbytes, int max_batch, char* err, size_t errlen);
void  dfo_free(dfo_model*);
void  dfo_set_threads(int n);                       /* OpenMP threads for the big loops (<=0: all) */
int   dfo_get_threads(void);
void  dfo_enable_taps(dfo_model*, int on);          /* allocate + record per-layer taps */
void  dfo_reset(dfo_model*, int seq);               /* seq < 0: all sequences */
int   dfo_step(dfo_model*, const int32_t* tokens, int batch);   /* 0 ok, <0 bad argument */
const float*   dfo_logits(const dfo_model*);        /* [batch][vocab] of the last step */
const int32_t* dfo_next_tokens(const dfo_model*);   /* [batch] */
const float*   dfo_hidden(const dfo_model*);        /* [batch][d_model] final residual (pre final norm) */
const void*    dfo_tap(const dfo_model*, int layer, int which, int seq, size_t* nbytes);
float* dfo_ssm_state(dfo_model*, int layer, int seq);   /* [nheads][headdim][d_state] */
float* dfo_conv_state(dfo_model*, int layer, int seq);  /* [conv_dim][3] */
int    dfo_shape(const dfo_model*, int32_t out[12]);    /* the header's 9 ints + nheads,d_in_proj,conv_dim */

/* fp16 state format (R24): binary32 -> binary16 RN-even, and the model switch (state rounded after every step) */
uint16_t dfo_float_to_half(float f);
void dfo_round_state_f16(float* H, size_t n);
void dfo_set_state_fp16(dfo_model*, int on);

/* temperature / top-k sampling of one token (R23); top_k <= 64 */
int dfo_sample(const float* logits, int n, float temperature, int top_k, float u);

/* TEST-ONLY arithmetic mode switch (see dfssm_oracle.c): the default is the contract. */
enum { DFO_MODE_CONTRACT = 0, DFO_MODE_REVERSED = 1, DFO_MODE_F64 = 2 };
void dfo_set_mode(int mode);
int dfo_get_mode(void);

#ifdef __cplusplus
}
#endif
#endif
