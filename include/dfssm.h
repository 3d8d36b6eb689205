/*
 * dfssm.h -- C ABI of the DF-SSM per-token decode step for one NVIDIA B200 (sm_100a).
 *
 * What the library computes (citations: "P:NN" = line NN of the paper text PAPER.md of
 * arxiv/paper_2606_10932; "R#" = a reading listed in DESIGN.md section 4):
 *
 *   for every sequence s of a batch, independently, with persistent per-sequence state,
 *     S0  u = e_s[tok] * float(E[tok,:])                       int8 per-row embedding
 *     for each layer:
 *     S1  RMSNorm(u) -> per-token absmax int8 (xq, s_x)        (R4, R13)
 *     S2  acc_i = sum_k sign_ik * xq_k, sign in {-1,+1}        bit-packed scaffold, int32
 *     S3  t_j = sum_k A_jk xq_k (int32);  zxbcdt_i = s_x*(w_s[i]*acc_i + b_s[i]*sum_j B_ij*(a_s[j]*t_j))
 *                                                              int8 LoRA, Eq. 3            (R5-R7)
 *     S4  causal depthwise 4-tap conv step over a rolling state, then SiLU   (R9)
 *     S5  h <- exp(dt*A)*h + (dt*x) (x) B ;  y = C.h + D*x     fp32 state                  (Table 12; R10-R12)
 *     S6  g = y*silu(z) ; RMSNorm(g) -> int8 (gq, s_g)         gate first, then norm
 *     S7  out_proj as S2/S3 on gq ; u <- u + out
 *     S8  RMSNorm(u) -> int8 ; logits_v = float(sum_k E_vk hq_k) * (s_h*e_s[v]) ; argmax (tied head; R16)
 *
 * Conventions
 *   - every function returns an int status (DFSSM_OK == 0, errors negative) unless stated;
 *     nothing throws, prints, or keeps global state; a handle is not thread-safe.
 *   - "dev" pointers are CUDA device pointers, "host" pointers are ordinary host pointers.
 *   - the CALLER owns the device arena, the CUDA stream and every host buffer; the LIBRARY
 *     owns what it places inside the arena and hands out BORROWED device pointers that stay
 *     valid until dfssm_destroy (their contents change at every dfssm_step).
 *   - all device work is enqueued on the stream given to dfssm_create; functions documented as
 *     "async" do not synchronise with the host.
 *   - there is no CPU fallback: on a device that is not compute capability 10.x
 *     dfssm_create fails with DFSSM_E_ARCH.
 */
#ifndef DFSSM_H
#define DFSSM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DFSSM_ABI_VERSION 1u

#if defined(__GNUC__)
#define DFSSM_API __attribute__((visibility("default")))
#else
#define DFSSM_API
#endif

enum {
    DFSSM_OK      = 0,
    DFSSM_E_ARG   = -1,   /* null pointer, batch out of range, bad index, unsupported shape */
    DFSSM_E_SIZE  = -2,   /* arena or blob too small / blob size does not match its header   */
    DFSSM_E_STATE = -3,   /* call out of order (step before load_weights, ...)               */
    DFSSM_E_CUDA  = -4,   /* a CUDA call failed; text in dfssm_last_error                    */
    DFSSM_E_ARCH  = -5,   /* device is not sm_100                                            */
    DFSSM_E_TOKEN = -6    /* a token id outside [0, vocab) was seen (it was clamped)          */
};

/* dfssm_config.flags */
#define DFSSM_FLAG_TAPS      1u  /* allocate per-layer debug taps and record them every step (slower)   */
#define DFSSM_FLAG_NO_GRAPH  2u  /* launch the step's kernels one by one instead of one CUDA-graph launch */
#define DFSSM_FLAG_NO_MEGA   4u  /* never use the single persistent kernel ("mega" path) for batch-1 steps    */
#define DFSSM_FLAG_NO_MMA   16u  /* keep the projections on the dp4a path at every batch size instead of tcgen05 kind::i8 tiles  */
#define DFSSM_FLAG_STATE_FP16 64u /* SURVEY 8(f) NEXT-2, first step (R24): the SSM state is STORED as binary16 (round to nearest even of each
                                   * step's binary32 update; the step's own readout uses the unrounded values).  Halves the state bytes (95 % of the
                                   * traffic at batch 64).  LOSSY against the fp32-state model; bit-identical to the oracle in the same mode.
                                   * Served by the kernel chain and dfssm_prefill (the persistent batch-1 kernel keeps fp32 state). */
#define DFSSM_FLAG_SCAFFOLD17 128u /* the blob holds the 17-level scaffold of PAPER.md Eq. 1 / Eq. 3 (weights level/8,
                                   * level in [-8, 8], five bit planes per 32 weights) instead of the 1-bit one; row scales apply to sum(level * q) */
#define DFSSM_FLAG_LORA_INT4 256u /* the blob holds int4 LoRA matrices (Table 4), two values per byte.
                                   * Both variants: the blob header's format word (offset 52: bit 0 / bit 1) must agree with these flags; served by
                                   * the kernel chain with tensor-core projections at every batch size and by dfssm_prefill; they need
                                   * d_model % 128 == 0, d_inner % 128 == 0 and lora_rank in {8, 16, 32, 64}, and exclude DFSSM_FLAG_NO_MMA. */
#define DFSSM_FLAG_PROF      8u  /* persistent kernel: thread 0 of every CTA stamps its SM clock at every phase */

/* Shape of the model (the paper's Mamba-2-shaped student, Table 1) + capacity.
 * nheads = d_inner/headdim ; d_in_proj = 2*d_inner + 2*ngroups*d_state + nheads ;
 * conv_dim = d_inner + 2*ngroups*d_state.  Requirements: d_model % 32 == 0, d_inner % 32 == 0,
 * d_inner % headdim == 0, nheads % ngroups == 0, d_conv == 4, d_state % 32 == 0, headdim % 16 == 0,
 * 1 <= lora_rank <= 64, d_model <= 8192, d_inner <= 8192, 1 <= max_batch <= 256. */
typedef struct dfssm_config {
    uint32_t abi_version;   /* DFSSM_ABI_VERSION */
    int32_t  n_layers, d_model, d_inner, headdim, d_state, ngroups, d_conv, vocab, lora_rank;
    int32_t  max_batch;     /* number of independent sequences the state is sized for */
    float    norm_eps;      /* RMSNorm epsilon (R13: 1e-5) */
    uint32_t flags;         /* DFSSM_FLAG_* */
} dfssm_config;

typedef struct dfssm_ctx dfssm_ctx;   /* opaque */

/* Debug taps (`which` of dfssm_debug_tensor), per layer and per sequence; recorded only with
 * DFSSM_FLAG_TAPS.  Same meaning as the rows of the step list above. */
enum {
    DFSSM_TAP_XQ_IN = 0,   /* int8  [d_model]    S1 codes                         */
    DFSSM_TAP_S_IN,        /* f32   [1]          S1 scale s_x                      */
    DFSSM_TAP_ACC_IN,      /* int32 [d_in_proj]  S2                                */
    DFSSM_TAP_T_IN,        /* int32 [lora_rank]  S3 stage 1                        */
    DFSSM_TAP_ZXBCDT,      /* f32   [d_in_proj]  S3 output, order z|x|B|C|dt       */
    DFSSM_TAP_XBC_CONV,    /* f32   [conv_dim]   S4 output (after SiLU)            */
    DFSSM_TAP_DT,          /* f32   [nheads]     softplus(dt_raw + dt_bias)        */
    DFSSM_TAP_Y,           /* f32   [d_inner]    S5 output                         */
    DFSSM_TAP_G,           /* f32   [d_inner]    y*silu(z)                         */
    DFSSM_TAP_GQ,          /* int8  [d_inner]    S6 codes                          */
    DFSSM_TAP_S_G,         /* f32   [1]          S6 scale                          */
    DFSSM_TAP_ACC_OUT,     /* int32 [d_model]    S7 scaffold                       */
    DFSSM_TAP_T_OUT,       /* int32 [lora_rank]  S7 LoRA stage 1                   */
    DFSSM_TAP_HIDDEN,      /* f32   [d_model]    residual stream after the layer   */
    DFSSM_TAP_COUNT
};

/* Device bytes the caller must provide for `cfg` (weights + per-sequence state + activations
 * [+ taps]).  Returns 0 if cfg is null or invalid. */
DFSSM_API size_t dfssm_arena_bytes(const dfssm_config* cfg);

/* Create a context on the CURRENT CUDA device.  dev_arena: device memory, 256-byte aligned,
 * at least dfssm_arena_bytes(cfg) bytes, owned by the caller and untouched by anyone else while
 * the context lives.  cuda_stream: a cudaStream_t (NULL = the legacy default stream).
 * The state is zeroed (as by dfssm_reset_state(ctx, -1)).  Synchronises the stream. */
DFSSM_API int dfssm_create(const dfssm_config* cfg, void* dev_arena, size_t arena_bytes, void* cuda_stream,
                 dfssm_ctx** out);

/* Load the canonical weight blob (layout: DESIGN.md section 3; header must match cfg).
 * host_blob is read during the call only.  Validates, copies to the arena, builds the per-layer
 * tables and the whole-step CUDA graph.  Synchronises the stream. */
DFSSM_API int dfssm_load_weights(dfssm_ctx* ctx, const void* host_blob, size_t nbytes);

/* Zero the conv + SSM state of sequence seq_index (or all sequences if < 0).  Async.
 * "State tensors ... are preallocated and persist across tokens". */
DFSSM_API int dfssm_reset_state(dfssm_ctx* ctx, int seq_index);

/* One decode step for sequences 0..batch-1: tokens_dev[s] is the input token of sequence s
 * (device int32[batch]; it may be the pointer returned by dfssm_next_tokens -- greedy decode
 * without leaving the device).  Async: for batch 1 exactly one launch of the persistent cooperative
 * kernel (the "mega" path: 148 co-resident CTAs, weights and state prefetched ahead of the layer
 * dependencies), for batch 2..3 of models with d_model >= 1024 one such launch per sequence, otherwise one CUDA graph of
 * the kernel chain, its kernels launched dependently (each runs its weight prologue while the one in front drains), with the
 * projections on tcgen05 kind::i8 tiles from batch 4 on (d_model >= 1024; from 2 on for d_model 512..1023, from 8 on below) -- unless
 * DFSSM_FLAG_NO_GRAPH or DFSSM_FLAG_TAPS asks for the chain's kernels one by one.  The paths share the state layout
 * and compute bit-identical results.  Token ids outside [0, vocab) are clamped on the
 * device and a sticky error is raised, reported as DFSSM_E_TOKEN by the next dfssm_sync. */
DFSSM_API int dfssm_step(dfssm_ctx* ctx, const int32_t* tokens_dev, int batch);

/* Prefill (the paper feeds prompts in chunks): feed n_tokens >= 1 prompt tokens
 * (device int32[n_tokens]) of ONE sequence `seq` in [0, max_batch).  Equivalent to n_tokens calls of dfssm_step for that
 * sequence alone -- bit-identical recurrent state, hidden state, logits and greedy token of the LAST position (readable
 * through dfssm_logits / dfssm_next_tokens / dfssm_hidden at index seq) -- but the projections run over up to 128 positions at a
 * time with the weights read once per chunk, and only the conv / state recurrence is serial in the position.  Async.
 * Shapes whose d_state is not a multiple of 16 (and contexts with DFSSM_FLAG_TAPS) are fed token by token instead (max_batch 1 only). */
DFSSM_API int dfssm_prefill(dfssm_ctx* ctx, const int32_t* tokens_dev, int n_tokens, int seq);

/* On-device temperature / top-k sampling (the generation loop of P:126; definition: DESIGN.md R23) from the
 * logits of the last step, for sequences 0..batch-1: the top_k (1..64) largest logits, equal logits by lower index first;
 * weights sp_expf((l - l_max) / temperature); the token whose running sum (binary64, rank order) first exceeds
 * uniform_dev[s] * total.  uniform_dev: device f32[batch], each in [0, 1) -- the caller's random numbers (the library draws none).
 * Overwrites the greedy tokens (dfssm_next_tokens), so feeding that pointer to the next dfssm_step decodes the sampled tokens
 * without leaving the device.  temperature <= 0 or top_k == 1 is greedy decode.  Async. */
DFSSM_API int dfssm_sample(dfssm_ctx* ctx, int batch, float temperature, int top_k, const float* uniform_dev);

/* Host-buffer form of the same step (the end-to-end call): copies tokens_host[batch] to the
 * device, runs the step, copies the greedy next tokens to next_host[batch] and, if logits_host is
 * non-null, the logits to logits_host[batch*vocab]; synchronises the stream before returning.
 * For best speed the host buffers should be page-locked; pageable memory also works. */
DFSSM_API int dfssm_step_host(dfssm_ctx* ctx, const int32_t* tokens_host, int batch, int32_t* next_host,
                    float* logits_host);

/* Borrowed device pointers to the results of the last step: logits f32 [batch][vocab] (row
 * stride = vocab), greedy tokens int32 [batch] (lowest index on ties), final residual stream
 * f32 [batch][d_model] (before the final norm).  No synchronisation: stream order applies. */
DFSSM_API int dfssm_logits(dfssm_ctx* ctx, const float** logits_dev);
DFSSM_API int dfssm_next_tokens(dfssm_ctx* ctx, const int32_t** next_dev);
DFSSM_API int dfssm_hidden(dfssm_ctx* ctx, const float** hidden_dev);

/* Borrowed device pointer + byte count of one debug tap of (layer, sequence).  DFSSM_E_STATE if
 * the context was created without DFSSM_FLAG_TAPS. */
DFSSM_API int dfssm_debug_tensor(dfssm_ctx* ctx, int layer, int which, int seq, const void** dev, size_t* nbytes);

/* Copy the recurrent state of (layer, seq) to / from HOST memory and synchronise.
 *   ssm  : f32 [nheads][headdim][d_state]   (may be null to skip)
 *   conv : f32 [conv_dim][3], oldest sample first   (may be null to skip)
 * The *_bytes arguments must equal the exact sizes (DFSSM_E_SIZE otherwise). */
DFSSM_API int dfssm_get_state(dfssm_ctx* ctx, int layer, int seq, float* ssm_host, size_t ssm_bytes,
                    float* conv_host, size_t conv_bytes);
DFSSM_API int dfssm_set_state(dfssm_ctx* ctx, int layer, int seq, const float* ssm_host, size_t ssm_bytes,
                    const float* conv_host, size_t conv_bytes);

/* In-kernel phase profile of the LAST persistent-kernel step (needs DFSSM_FLAG_PROF; a tracing aid, not
 * part of the method).  dims[3] receives {CTAs, layers + 1, stamps per (CTA, layer)}; if stamps_host is
 * non-null it must hold exactly CTAs*(layers+1)*stamps uint64 (nbytes), filled with the SM-clock value
 * (clock64) thread 0 of each CTA read at each phase boundary of each layer; stamp 15 is %globaltimer (ns) at
 * the start of the layer; row `layers` is the LM head (stamps 0, 1).  Synchronises the stream. */
DFSSM_API int dfssm_debug_profile(dfssm_ctx* ctx, uint64_t* stamps_host, size_t nbytes, int32_t* dims);

/* Wait for the stream; returns DFSSM_E_TOKEN once if a bad token id was clamped since the last
 * call, DFSSM_E_CUDA on a device fault or if a step timed out on the device (an exchange between the
 * CTAs of the persistent kernel, or a tensor-core projection, did not complete within ~0.3 s).  After
 * such a time-out the recurrent state is half-written: dfssm_step returns DFSSM_E_STATE until
 * dfssm_reset_state(ctx, -1) has been called. */
DFSSM_API int dfssm_sync(dfssm_ctx* ctx);

/* Number of kernels of this library that one dfssm_step(batch) launches (graph nodes).  >= 1. */
DFSSM_API int dfssm_launches_per_step(dfssm_ctx* ctx, int batch);

/* Device-timed profile of the last `dfssm_step` when run with per-kernel events is not offered;
 * use dfssm_time_kernels: runs `iters` steps with CUDA events around every kernel class and
 * writes the mean microseconds per step of each class to out_us[DFSSM_KCLASS_COUNT].  Sync. */
enum {
    DFSSM_KCLASS_EMBED = 0, DFSSM_KCLASS_NORMQUANT, DFSSM_KCLASS_PROJ_IN, DFSSM_KCLASS_SSM,
    DFSSM_KCLASS_PROJ_OUT, DFSSM_KCLASS_EPI_OUT, DFSSM_KCLASS_LMHEAD, DFSSM_KCLASS_ARGMAX,
    DFSSM_KCLASS_MEGA,     /* the whole step as one persistent kernel (batch 1); the others are then 0 */
    DFSSM_KCLASS_COUNT
};
DFSSM_API int dfssm_time_kernels(dfssm_ctx* ctx, const int32_t* tokens_dev, int batch, int iters,
                       float* out_us /* [DFSSM_KCLASS_COUNT] */);

/* Human-readable text for the last error of this context ("" if none).  Never null. */
DFSSM_API const char* dfssm_last_error(const dfssm_ctx* ctx);

/* Release the context (never frees the arena).  Safe on null. */
DFSSM_API void dfssm_destroy(dfssm_ctx* ctx);

/* ---- Continuous-batching greedy generator (second half; the generation loop of P:126) ----------------------
 * Host logic over ONE context (paper_2606_10932_b200/csrc/dfssm_sched.cu; no kernel of its own): requests wait in a FIFO; every
 * iteration admits waiting requests into free sequence slots (lowest first: dfssm_reset_state + dfssm_prefill of the prompt, which
 * leaves the request's first generated token in the context's token buffer), runs ONE dfssm_step for slots 0 .. highest active
 * slot with that device buffer as input, reads the new tokens back and retires finished requests.  Sequences are independent in
 * every kernel, so a request's tokens equal those of running it alone, whatever the schedule.  One scheduler per context; N GPUs =
 * N contexts + N schedulers fed by the caller (replicas only).
 *   dfssm_sched_create   ctx: a loaded context whose max_batch >= max_batch; dev_scratch: caller-owned device memory that holds one
 *                        prompt at a time and max_batch uniforms (scratch_bytes / 4 - max_batch = the longest prompt accepted);
 *                        cuda_stream: the CONTEXT's stream.
 *   dfssm_sched_submit   copies the prompt (host int32[n_prompt], n_prompt >= 1) and queues it; *request_id = its handle.
 *   dfssm_sched_iterate  one iteration as above; *n_active = requests generating or waiting afterwards.  Synchronises the stream.
 *   dfssm_sched_run      iterates until nothing is active, then dfssm_sync (DFSSM_E_TOKEN if a prompt held a bad token id).
 *   dfssm_sched_result   the tokens generated so far for a request (copied to tokens_host[capacity] if given), *done = finished.
 *   dfssm_sched_stats    steps run, and slot-steps used by live requests / run in total (idle slots below the highest live one).
 * The context must not be stepped by anyone else while a scheduler drives it.  Errors as for the calls it makes. */
typedef struct dfssm_sched dfssm_sched;
DFSSM_API int dfssm_sched_create(dfssm_ctx* ctx, int max_batch, void* dev_scratch, size_t scratch_bytes, void* cuda_stream, dfssm_sched** out);
DFSSM_API int dfssm_sched_submit(dfssm_sched* s, const int32_t* prompt_host, int n_prompt, int max_new_tokens, int* request_id);
/* Sampled instead of greedy generation (only while no request is generating): one temperature / top_k (1..64) for the scheduler
 * (temperature <= 0 or top_k == 1: greedy); token k (0-based) of request id is drawn by dfssm_sample with the uniform
 * dfssm_sched_uniform(seed + id, k), a counter-based generator (splitmix64 finaliser of seed' + (k + 1) * 0x9E3779B97F4A7C15; its top
 * 24 bits / 2^24, in [0, 1)), so a request's tokens do not depend on the schedule.  The last max_batch words of dev_scratch hold
 * the uniforms: the longest prompt accepted is scratch_bytes / 4 - max_batch. */
DFSSM_API int dfssm_sched_set_sampling(dfssm_sched* s, float temperature, int top_k, unsigned long long seed);
DFSSM_API float dfssm_sched_uniform(unsigned long long seed, int k);
DFSSM_API int dfssm_sched_iterate(dfssm_sched* s, int* n_active);
DFSSM_API int dfssm_sched_run(dfssm_sched* s);
DFSSM_API int dfssm_sched_result(dfssm_sched* s, int request_id, int32_t* tokens_host, int capacity, int* n_tokens, int* done);
DFSSM_API int dfssm_sched_stats(dfssm_sched* s, long long* steps, long long* slot_steps_used, long long* slot_steps_run);
DFSSM_API const char* dfssm_sched_last_error(const dfssm_sched* s);
DFSSM_API void dfssm_sched_destroy(dfssm_sched* s);

/* ---- S8 without any allocation, context or arena (paper_2606_10932_b200/csrc/dfssm_noalloc.cu) -------------------------------
 * For callers that cannot call cudaMalloc and cannot hand over an arena (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid allocation).  Computes, for `batch` sequences, what the end of dfssm_step computes (S8: PAPER.md P:96,
 * DESIGN.md R16, R19): final RMSNorm + absmax int8 quantiser of the hidden state, tied int8 LM head
 * logit_v = float(sum_k E_vk q_k) * (s_h * e_s[v]), greedy token = argmax with the lowest index on ties.  Bit-identical to
 * dfssm_step's logits and tokens for the same hidden state and weights.
 *   hidden_dev      device, float [batch][d_model]           (e.g. dfssm_hidden)            read
 *   normf_w_dev     device, float [d_model]                  final norm weight              read
 *   emb_dev         device, int8  [vocab][d_model], 16-byte aligned; emb_scale_dev device float [vocab]   read
 *   next_dev        device, int32 [batch]                    greedy tokens                  written
 *   logits_dev      device, float [batch][vocab] or NULL     copy of the logits             written if given
 *   cuda_stream     cudaStream_t (0 = the default stream); the three kernels are enqueued on it, nothing is synchronised
 * All buffers are the caller's.  The intermediates (codes, scales, logits) live in a static device array of
 * DFSSM_NOALLOC_SCRATCH_BYTES that every GPU holds from the moment libdfssm.so is loaded until the process exits; a call needs
 * dfssm_head_noalloc_scratch_need(batch, d_model, vocab) = up256(batch*d_model) + up256(4*batch) + 4*batch*vocab bytes of it
 * (cfg 2: batch <= 20) and is rejected with DFSSM_E_SIZE beyond that.  Calls no cudaMalloc / cudaFree / allocating routine.
 * The first call on a device takes the array's address (cudaGetSymbolAddress, that device current); later calls only launch.
 * EVERY call on a device shares the array and finds the previous call's contents in it (nothing needs clearing: every value
 * read is written earlier in the same call).  Calls that overlap on the GPU (different streams without an ordering between
 * them) RACE on it: keep them on one stream or order them with events.
 * Errors: DFSSM_E_ARG (null pointer, batch / vocab < 1, d_model not a positive multiple of 16 or > 6144, misaligned emb_dev),
 * DFSSM_E_SIZE (scratch), DFSSM_E_ARCH (not sm_100), DFSSM_E_CUDA; text from dfssm_head_noalloc_error (per host thread). */
#define DFSSM_NOALLOC_SCRATCH_BYTES (4u << 20)
DFSSM_API size_t dfssm_head_noalloc_scratch_need(int batch, int d_model, int vocab);
DFSSM_API int dfssm_head_noalloc(const float* hidden_dev, const float* normf_w_dev, const int8_t* emb_dev, const float* emb_scale_dev,
                                 int batch, int d_model, int vocab, float eps, int32_t* next_dev, float* logits_dev, void* cuda_stream);
DFSSM_API const char* dfssm_head_noalloc_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DFSSM_H */
