// "mega" path: the whole decode step of ONE sequence (S0, L x (S1..S7), S8) as ONE persistent
// cooperative kernel, one CTA per SM.  (the paper removes launch overhead with a CUDA graph;
// here the step is a single launch and the per-layer dependencies are resolved inside the kernel.)
//
// Design:
//   * Roles.  The 148 CTAs are NW "workers" (CTAs 0 .. NW-1) and NS = 148 - NW "service" CTAs.
//     Worker c owns d_inner channels [chs[c], chs[c+1]) -- their z and x in_proj rows, their conv and SSM
//     state, their gate -- and out_proj rows [ors[c], ors[c+1]) with that slice of the residual stream u (kept
//     in shared memory for the whole step).  The service CTAs own the rows whose result EVERY worker needs and
//     that need the whole activation vector: the B|C|dt in_proj rows and the LoRA down-projections t = A.xq of
//     both projections.  They own no state and stream almost no weights, so they are always waiting when an
//     activation vector completes and publish their few int32 words while the workers are still busy with
//     their own sign rows: the two small exchanges (A, T) overlap with the workers' integer work instead of
//     following it (round 1 dealt these rows round-robin over all CTAs: every worker then waited for the
//     slowest of 148 publishers, 2.5 k + 1.7 k clocks per layer).
//   * Weights.  dfssm_load_weights repacks every layer into one contiguous chunk per (layer, worker)
//     (sign rows, LoRA-up rows, scales, conv taps, per-channel constants), one chunk per (layer, service CTA)
//     (its sign rows and LoRA-down rows) plus one block per layer that every worker reads (the LoRA-up rows /
//     scales / conv taps of the B|C|dt rows).  Chunk + block + the CTA's slice of the SSM / conv state form one
//     pipeline item, fetched by bulk async copies (cp.async.bulk -> mbarrier) into a ring of shared-memory
//     stages several layers AHEAD of the dependency chain: addresses never depend on activations, so HBM stays
//     busy while CTAs wait on each other.  The LM head streams the int8 embedding through the same ring.
//   * Exchange.  Four self-validating all-gathers per layer through L2:
//       U : t_k = u_k * w_k (fp32) of the owned out rows (+ the worker's partial sum of u^2, fp64, in its own array)
//           -> every CTA derives amax and the int8 codes of the WHOLE vector itself (S1)
//       A : raw int32 accumulators of the B|C|dt rows + t_in   (service -> workers)
//           -> every worker finishes the B|C|dt epilogue, conv and softplus itself (S3, S4)
//       G : t_k = g_k * w_k (fp32) of the owned channels (+ partial sum of g^2)  -> S6 everywhere
//       T : partial LoRA-down sums of out_proj                 (service -> workers)
//     Every 32-bit word is either the sentinel 0xffffffff or payload (fp32 values are never that NaN; int32
//     values are stored with the sign bit flipped; fp64 partials are 8-byte stores validated by their high
//     word), so a hop is one store and one successful poll: no flag, no fence.
//   * Memory ordering (PTX model).  There are 2 x L records: step n publishes layer l into record (n & 1, l) and
//     resets its own words of record (~n & 1, l) to the sentinel.  Inside one launch a word is therefore written
//     ONCE and never reset, and a word that is reset is never polled: every reset is ordered against the polls
//     that need it, and against the reads that precede it, by a KERNEL BOUNDARY (the record was last read by
//     the previous launch and is next polled by the following one).  All exchange accesses are relaxed gpu-scope
//     64-bit accesses (single-copy atomic, "morally strong": no data race); a poll accepts only a non-sentinel
//     value, which can only be this launch's payload.  No ordering rests on elapsed time, and no fence is needed
//     (round 1 rotated 4 records inside a launch and relied on a reset being "at least two hops old";
//     fence.acq_rel.gpu around every publish and gather was measured at ~1000 clocks per fence, +55 % step time).
//   * Critical path.  Only amax -> 127/amax -> codes is on it; the fp64 sum of squares, rstd and the activation
//     scale are made by one warp from the partial array while the sign rows run (they are first needed in the
//     projection epilogue).
//   * Arithmetic: identical to the chain path (dfssm_math.cuh; contract of DESIGN.md section 5).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "dfssm_kernels.cuh"
#include "dfssm_math.cuh"

namespace dfssm {
namespace mega {

#ifndef DFSSM_THREADS
#define DFSSM_THREADS 512
#endif
constexpr int THREADS = DFSSM_THREADS;        // 16 or 32 warps
constexpr int NWARPS = THREADS / 32;
constexpr int NJ_MAX = 3072 / THREADS;        // 16-byte chunks per thread when gathering U / G with run-time shapes (plan() checks)
constexpr int NJ_A = 1024 / THREADS;          // ... when gathering A
constexpr int NR_IN = THREADS >= 1024 ? 2 : 4;     // in_proj sign rows per warp pass
constexpr int LPC = THREADS / 32;             // lanes per channel in the state update (32 channels per pass)
constexpr int LPB = THREADS / 512;            // lanes per B|C row in the in_proj epilogue
constexpr int SCALE_WARP = 0;                 // the warp of the scale CTA that finishes the activation scales
constexpr int DMA_TID = 96;                   // the thread that issues the state write-back and the ring refills (a warp off the publish paths)
constexpr int KS_MAX = 4;                     // largest K-split of the out_proj sign rows
constexpr int MAX_STAGES = 8;
constexpr uint32_t SPIN_LIMIT = 1u << 20;     // ~0.3 s of polling, then the step aborts with an error flag
constexpr uint32_t SENT = 0xffffffffu;        // "not written yet"
constexpr uint32_t IBIAS = 0x80000000u;       // int32 payloads are stored xor IBIAS (|value| < 2^30)
constexpr int PROF_NPH = 32;                  // phase stamps per (CTA, layer) of the in-kernel profiler

constexpr int GRID = 148;                     // one CTA per B200 SM
constexpr int NW_CT = 128;                    // workers of the compile-time-shape kernels (the rest are service CTAs)

// mailboxes of the small parts A and T (each must divide GRID and be <= MBOX): the payload is pushed M times and GRID / M
// workers poll each copy (polls that reach a line before the data delay the stores to it).  U and G have one copy.
#ifndef DFSSM_MA
#define DFSSM_MA 1
#endif
#ifndef DFSSM_MT
#define DFSSM_MT 1
#endif
// clocks a worker waits after publishing G / U before its first poll (round 1: polls that reach a line before the data delay
// the stores to it, 500 clocks paid; with 128-byte-aligned full slots and the resets moved behind the publish: 0 / 250 / 500
// clocks -> 389.6 / 392.7 / 399.0 us per step, so no wait)
#ifndef DFSSM_WG
#define DFSSM_WG 0
#endif
#ifndef DFSSM_WU
#define DFSSM_WU 0
#endif
constexpr int MBOX = DFSSM_MA > DFSSM_MT ? DFSSM_MA : DFSSM_MT;      // small mailboxes allocated per record
constexpr int M_A = DFSSM_MA, M_T = DFSSM_MT;

struct Params {
    // ---- shape ----
    int L, d_model, d_inner, headdim, d_state, ngroups, nheads, r, vocab, n_bcdt, gs;
    float eps;
    int G, NW, NS, NT;           // grid size (all co-resident), workers, service CTAs, of which NT = NS - 1 hold row tasks
    int nch_max, nor_max, r_pad;
    int Win, Wout;               // sign words per row of in_proj / out_proj
    int n_early;                 // service results of in_proj: n_bcdt sign rows + r LoRA-down rows
    int tsplit, n_ttask;         // out_proj LoRA-down rows are split into tsplit partial tasks each
    int ns_sig, ns_lin, ns_tt;   // most sign rows / in_proj LoRA-down rows / out_proj partial tasks one service CTA holds
    // ---- worker chunk layout (byte offsets inside one (layer, worker) chunk) ----
    uint32_t c_in_bits, c_out_bits, c_in_B, c_out_B, c_in_scale, c_in_bs, c_out_scale, c_out_bs, c_conv_w, c_conv_b,
        c_alog, c_D, c_gnorm, c_nnorm, chunk_bytes;
    // ---- service chunk layout (byte offsets inside one (layer, service CTA) chunk) ----
    uint32_t sc_sign, sc_tin, sc_tout, schunk_bytes;
    // ---- per-layer block read by every worker (byte offsets) ----
    uint32_t b_eB, b_escale, b_ebs, b_econv_w, b_econv_b, b_dtb, b_as_in, b_as_out, blk_bytes;
    // ---- pipeline stage ----
    uint32_t st_blk, st_ssm, st_conv, st_econv, stage_bytes;
    int stages, lm_rows_item;
    // ---- exchange: 2 sets x L records; a record = main part (U, PU, G, PG: one copy) + MBOX small mailboxes (A, T);
    //      32-bit word offsets inside the main part / inside one small mailbox ----
    int u_slot, g_slot;          // words per worker slot of U / G (a power of two >= the owned elements)
    uint32_t x_U, x_PU, x_G, x_PG, x_main, x_A, x_T, x_small;      // PU / PG: the workers' fp64 partial sums of squares
    // ---- shared memory carve ----
    uint32_t s_ring, s_mbar, s_xq, s_bc, s_cd, s_u, s_z, s_x, s_dt, s_v, s_eacc, s_acc_in, s_acc_out, s_chs, s_ors,
        s_red, s_slot, s_scal, smem_bytes;
    // ---- device pointers ----
    const uint8_t* chunks;       // [L][NW][chunk_bytes]
    const uint8_t* schunks;      // [L][NT][schunk_bytes]
    const uint8_t* blocks;       // [L][blk_bytes]
    float* ssm;                  // sequence 0 of layer 0; layer stride ssm_lstride floats
    float* conv;                 // [conv_dim][4] ring of sequence 0 of layer 0; layer stride conv_lstride floats
    size_t ssm_lstride, conv_lstride;
    const int8_t* emb; const float* emb_s; const float* first_norm_w;
    const int32_t* tokens; int32_t* next; int32_t* tok_out; int32_t* pos;
    float* logits; float* u_out;
    uint32_t* xbuf;              // [2 sets][L][x_main + MBOX * x_small]
    float* am_val; int* am_idx; unsigned* am_count;
    int* err;
    uint32_t set;                // record set this step publishes into (step counter & 1); it resets the other one
    uint8_t* taps; size_t tap_lstride; TapLayout tl;
    unsigned long long* prof;    // [G][L+1][PROF_NPH] SM-clock stamps of thread 0 (DFSSM_FLAG_PROF), else null
};

// ------------------------------------------------------------------------------------------------
// PTX helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// the same copies with an L2 evict-first policy: weights and state are touched once per token and must not push the
// exchange mailboxes (polled every layer) or the per-layer shared blocks out of L2
__device__ __forceinline__ uint64_t policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void bulk_g2s_stream(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_s2g_stream(void* dst, const void* src_smem, uint32_t bytes, uint64_t pol)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst), "r"(smem_u32(src_smem)), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src_smem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// exchange words: relaxed gpu-scope accesses (served by L2; a 32-bit / 64-bit scalar access is single-copy atomic).
__device__ __forceinline__ void x_st32(uint32_t* p, uint32_t v)
{
    asm volatile("st.relaxed.gpu.global.b32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void x_st64(uint32_t* p, uint32_t lo, uint32_t hi)
{
    const uint64_t a = ((uint64_t)hi << 32) | lo;
    asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(p), "l"(a) : "memory");
}
// 16 bytes as TWO 64-bit elements, each single-copy atomic (a float pair, or one fp64)
__device__ __forceinline__ uint4 x_ld128(const uint32_t* p)
{
    uint64_t a, b;
    asm volatile("ld.relaxed.gpu.global.v2.b64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
    return make_uint4((uint32_t)a, (uint32_t)(a >> 32), (uint32_t)b, (uint32_t)(b >> 32));
}
__device__ __forceinline__ void x_st128(uint32_t* p, uint4 v)
{
    const uint64_t a = ((uint64_t)v.y << 32) | v.x, b = ((uint64_t)v.w << 32) | v.z;
    asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1,%2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
// Code layout for the masked-dp4a sign dot: a 32-block of codes is eight 4-byte words ("planes"), plane i = elements
// 4i .. 4i+3 of the block; the load-time repack moves the sign bit of element 4i + j to bit 8j + i of the sign word,
// so dp4a(bits & (0x01010101 << i), plane i) sums plane i.  Planes 0..3 of all blocks form the first half of
// the vector (16 B per block), planes 4..7 the second half: position of canonical element k in a vector of length K.
__device__ __forceinline__ int plane_pos(int k, int K)
{
    return ((k & 16) ? (K >> 1) : 0) + ((k >> 5) << 4) + (k & 15);
}

// Shape of the model as the kernel sees it: compile-time constants for the shapes of BASELINE.json's configs (every
// index computation, division and loop bound folds), or the run-time values of Params (any other shape).
struct ShapeRT { static constexpr bool kStatic = false; static constexpr int d_model = 0, d_inner = 0, headdim = 0, d_state = 0, ngroups = 0, r = 0, NW = 0; };
template <int DM, int DI, int HD, int DS, int NG, int R>
struct ShapeCT { static constexpr bool kStatic = true; static constexpr int d_model = DM, d_inner = DI, headdim = HD, d_state = DS, ngroups = NG, r = R, NW = NW_CT; };

// Ownership: worker g owns elements [own_start(g, n, NW), own_start(g + 1, n, NW)) of a vector of length n (n % 4 == 0),
// in groups of 4 so that a gathered 16-byte chunk is four consecutive elements of one 16-element half block of codes.
__host__ __device__ constexpr int own_start(int g, int n, int NW) { return 4 * (int)(((long long)g * (n / 4)) / NW); }
__host__ __device__ constexpr int own_max(int n, int NW) { return 4 * ((n / 4 + NW - 1) / NW); }
// words of one worker's slot in a U / G mailbox: a power of two (4, 8, 16 ...), so that a slot never straddles a 128-byte
// line (measured: 80-byte slots cost ~1000 clocks per hop more than 64- or 128-byte ones)
__host__ __device__ constexpr int slot_words(int need) { int w = 4; while (w < need) w *= 2; return w; }
// 16-byte chunks per thread needed to gather the NW slots of a vector of length n
__host__ __device__ constexpr int nj_slots(int n, int NW) { return (NW * slot_words(own_max(n, NW)) / 4 + THREADS - 1) / THREADS; }
// service CTA s holds the items s, s + NS, s + 2 NS ... of a list of n
__host__ __device__ constexpr int dealt(int n, int s, int NS) { return s < n ? (n - s + NS - 1) / NS : 0; }

template <class S>
struct Ctx {
    const Params& P;
    uint8_t* sm;
    int tid, lane, wid, c;
    volatile int* dead;          // shared flag: a poll timed out -> stop spinning everywhere
    bool prof;                   // in-kernel profiler on (a compile-time false in the production instantiations)
    static constexpr int NJG = S::kStatic ? nj_slots(S::d_inner, S::NW) : NJ_MAX;     // chunks per thread: gather G, gather U
    static constexpr int NJU = S::kStatic ? nj_slots(S::d_model, S::NW) : NJ_MAX;
    static constexpr int NJ0 = S::kStatic ? (S::d_model / 4 + THREADS - 1) / THREADS : 8192 / 4 / THREADS;   // embedding
    // every worker owns the same number of channels / out rows (a compile-time constant), and a slot holds exactly that many
    // words: element k of the gathered vector sits in chunk k / 4 (no ownership tables on the critical path)
    static constexpr bool kEven = S::kStatic && (S::d_inner / 4) % (S::kStatic ? S::NW : 1) == 0 && (S::d_model / 4) % (S::kStatic ? S::NW : 1) == 0;
    static constexpr int kNch = kEven ? S::d_inner / (S::kStatic ? S::NW : 1) : 0, kNor = kEven ? S::d_model / (S::kStatic ? S::NW : 1) : 0;
    static constexpr bool kDenseG = kEven && slot_words(kNch) == kNch, kDenseU = kEven && slot_words(kNor) == kNor;
#define DFSSM_DIM(n_) __device__ __forceinline__ int n_() const { return S::kStatic ? S::n_ : P.n_; }
    DFSSM_DIM(d_model) DFSSM_DIM(d_inner) DFSSM_DIM(headdim) DFSSM_DIM(d_state) DFSSM_DIM(ngroups) DFSSM_DIM(r) DFSSM_DIM(NW)
#undef DFSSM_DIM
    __device__ __forceinline__ void stamp(int l, int k) const
    {
        if (prof && tid == 0) {     // the clock is read behind a shared-memory load: a stamp after a barrier is the RELEASE time
            const int v = *dead;
            unsigned long long t;
            asm volatile("mov.u64 %0, %%clock64;" : "=l"(t) : "r"(v) : "memory");
            P.prof[((size_t)c * (P.L + 1) + l) * PROF_NPH + k] = t;
        }
    }
    __device__ __forceinline__ void gstamp(int l, int k) const      // %globaltimer (ns, one clock for all SMs): cross-CTA timelines
    {
        if (prof && tid == 0) {
            const int v = *dead;
            unsigned long long t;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t) : "r"(v) : "memory");
            P.prof[((size_t)c * (P.L + 1) + l) * PROF_NPH + k] = t;
        }
    }
    __device__ __forceinline__ constexpr int G() const { return GRID; }
    __device__ __forceinline__ int NS() const { return GRID - NW(); }
    __device__ __forceinline__ bool service() const { return c >= NW(); }
    __device__ __forceinline__ int nheads() const { return d_inner() / headdim(); }
    __device__ __forceinline__ int gs() const { return ngroups() * d_state(); }
    __device__ __forceinline__ int n_bcdt() const { return 2 * gs() + nheads(); }
    __device__ __forceinline__ int nch_max() const { return own_max(d_inner(), NW()); }
    __device__ __forceinline__ int nor_max() const { return own_max(d_model(), NW()); }
    __device__ __forceinline__ int r_pad() const { return (r() + 3) / 4 * 4; }
    __device__ __forceinline__ int Win() const { return d_model() / 32; }
    __device__ __forceinline__ int Wout() const { return d_inner() / 32; }
    __device__ __forceinline__ int n_early() const { return n_bcdt() + r(); }
    __device__ __forceinline__ int tsplit() const { return d_inner() % 64 == 0 ? 4 : 2; }
    __device__ __forceinline__ int n_ttask() const { return r() * tsplit(); }
    // words of the A / T part: the service results plus the activation scale(s) made by service CTA 0
    __device__ __forceinline__ int n_A() const { return n_early() + 1; }          // [n_early]: scale of this layer's in_proj codes
    __device__ __forceinline__ int i_sg() const { return (n_ttask() + 3) / 4 * 4; }   // T word: scale of this layer's out_proj codes (own chunk)
    __device__ __forceinline__ int i_slm() const { return i_sg() + 4; }               // T word: scale of the LM-head codes (last layer only; own chunk)
    __device__ __forceinline__ int u_slot() const { return slot_words(nor_max()); }
    __device__ __forceinline__ int g_slot() const { return slot_words(nch_max()); }
};

__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
// in-kernel profiler: thread 0 of every CTA stamps its SM clock at phase k of layer l
#define DFSSM_STAMP(l_, k_) x.stamp((l_), (k_))

template <class S>
__device__ __forceinline__ void poll_fail(const Ctx<S>& x)
{
    *x.dead = 1;
    atomicOr(x.P.err, 2);
}

// mailbox (of a part pushed M times) that CTA c polls, and the number of mailboxes the CTAs [0, n) poll
__device__ __forceinline__ constexpr int mbox_of(int c, int M) { return c / (GRID / M); }
__device__ __forceinline__ constexpr int mbox_count(int n, int M) { return (n + GRID / M - 1) / (GRID / M); }

// ------------------------------------------------------------------------------------------------
// exchange: gather a self-validating buffer
// ------------------------------------------------------------------------------------------------
// spin on ONE exchange word until it has been written
template <class S>
__device__ __forceinline__ uint32_t poll_word(const Ctx<S>& x, const uint32_t* w)
{
    uint32_t v, spins = 0;
    for (;;) {
        asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(w) : "memory");
        if (v != SENT) break;
        if (++spins > SPIN_LIMIT || *x.dead) { poll_fail(x); break; }
    }
    return v;
}

// scratch inside s_red: NWARPS doubles (warp sums of squares)
template <class S>
__device__ __forceinline__ double* red_d(const Ctx<S>& x) { return (double*)(x.sm + x.P.s_red); }
// a 16-byte chunk is complete when none of its four words is the sentinel (every part is padded to whole chunks and
// pad words hold 0 from load time on)
__device__ __forceinline__ bool chunk_ok(uint4 v) { return max(max(v.x, v.y), max(v.z, v.w)) != SENT; }

// Thread t owns the 16-byte chunks t, t + THREADS, ... (at most NJ) of the nchunk chunks at buf.  Spins until every owned
// word has been written; the raw words come back in v[].  tix = the thread's index for the chunk ownership (tid, or
// reversed so that the small gathers are polled by the warps that have nothing else to do).
// If `part` is given (the scale CTA gathering U or G), the lanes 0 .. PLN-1 of every warp also poll one chunk (two fp64 partial
// sums of squares, validated by their high words) of the workers' partial array, and the warp's sum of them is left in
// red_d[warp] (read by scale_finish behind the barriers of absmax_quant).
constexpr int PLN = 8;
template <int NJ, class S>
__device__ __forceinline__ void hop_gather(const Ctx<S>& x, const uint32_t* buf, int nchunk, uint4 (&v)[NJ], int tix, int first_wait = 0,
                                           const uint32_t* part = nullptr)
{
    bool need[NJ];
    bool any = false;
#pragma unroll
    for (int j = 0; j < NJ; ++j) { need[j] = tix + j * THREADS < nchunk; any = any || need[j]; }
    const int pch = x.wid * PLN + x.lane;
    bool needp = part != nullptr && x.lane < PLN && 2 * pch < x.NW();
    const bool hasp = needp;
    uint4 pv = make_uint4(0u, 0u, 0u, 0u);
    if (any || needp) {
        if (first_wait > 0) {                          // polls that arrive before the data delay the stores to the same lines
            const long long t0 = clock64();
            while (clock64() - t0 < first_wait) {}
        }
        uint32_t spins = 0;
        for (;;) {
#pragma unroll
            for (int j = 0; j < NJ; ++j)
                if (need[j]) v[j] = x_ld128(buf + 4 * (tix + j * THREADS));
            if (needp) pv = x_ld128(part + 4 * pch);
            bool all = true;
#pragma unroll
            for (int j = 0; j < NJ; ++j)
                if (need[j]) { need[j] = !chunk_ok(v[j]); all = all && !need[j]; }
            if (needp) { needp = pv.y == SENT || (2 * pch + 1 < x.NW() && pv.w == SENT); all = all && !needp; }
            if (all) break;
            if (++spins > SPIN_LIMIT || *x.dead) { poll_fail(x); break; }
        }
    }
    if (part != nullptr) {                             // warp-uniform
        double ps = 0.0;
        if (hasp) {
            ps = __hiloint2double((int)pv.y, (int)pv.x);
            if (2 * pch + 1 < x.NW()) ps += __hiloint2double((int)pv.w, (int)pv.z);
        }
        static_assert(PLN == 8, "three shuffle steps");
        ps += __shfl_xor_sync(0xffffffffu, ps, 1);
        ps += __shfl_xor_sync(0xffffffffu, ps, 2);
        ps += __shfl_xor_sync(0xffffffffu, ps, 4);
        if (x.lane == 0) red_d(x)[x.wid] = ps;
    }
}

// scalars: [0] amax of the last absmax_quant, [1] scale of the in_proj / LM-head codes, [2] scale of the out_proj codes;
// behind them the accumulators of the CTA-wide reductions, double-buffered by call parity: uint amax bits [2], int code sums [2]
template <class S>
__device__ __forceinline__ float* scal(const Ctx<S>& x) { return (float*)(x.sm + x.P.s_scal); }
template <class S>
__device__ __forceinline__ unsigned* acc_amax(const Ctx<S>& x) { return (unsigned*)(x.sm + x.P.s_scal) + 4; }
template <class S>
__device__ __forceinline__ int* acc_qs(const Ctx<S>& x) { return (int*)(x.sm + x.P.s_scal) + 6; }

// S1 / S6 / S8 absmax + quantise of a whole vector in every CTA (the critical path of the norm: only amax is needed for
// the codes, R13).  `en(f)` calls f(k, bits) for every group of four elements this thread holds: bits = fp32 t_k = value_k * w_k.
// Writes the codes to xq (plane order unless `canonical`), leaves amax in scal[0] and returns the sum of the codes.
// The two CTA-wide reductions (max, integer sum: exact in any order) are shared-memory atomics into accumulators that
// alternate with the call parity `par`; thread 0 clears the other pair between the two barriers.  Two __syncthreads.
// (Tried: every warp polls a 512-byte array of the workers' own maxima and skips the first barrier -- 2368 warps then hammer
// four L2 lines and the gathers go from 1.0 k to 9.5 k clocks.)
template <class S, typename Enum>
__device__ __forceinline__ int absmax_quant(const Ctx<S>& x, Enum en, int K, bool canonical, int8_t* tap_codes, unsigned& par,
                                          int pl = 0, int pk = -1)
{
    const Params& P = x.P;
    uint8_t* xq = x.sm + P.s_xq;
    unsigned am = 0u;                  // |t| as bits: non-negative floats order like unsigned integers
    en([&](int, uint4 w) { am = max(max(am, w.x & 0x7fffffffu), max(max(w.y & 0x7fffffffu, w.z & 0x7fffffffu), w.w & 0x7fffffffu)); });
    am = __reduce_max_sync(0xffffffffu, am);
    if (x.lane == 0) atomicMax(acc_amax(x) + par, am);
    if (pk >= 0) x.stamp(pl, pk);
    __syncthreads();
    if (pk >= 0) x.stamp(pl, pk + 1);
    const float amax = __uint_as_float(acc_amax(x)[par]);
    const float inv = amax == 0.0f ? 0.0f : fdiv(127.0f, amax);
    int qs = 0;
    en([&](int k0, uint4 w) {                                       // four consecutive elements, k0 % 4 == 0
        const uint32_t q0 = (uint32_t)quant_code(__uint_as_float(w.x), inv) & 255u, q1 = (uint32_t)quant_code(__uint_as_float(w.y), inv) & 255u,
                       q2 = (uint32_t)quant_code(__uint_as_float(w.z), inv) & 255u, q3 = (uint32_t)quant_code(__uint_as_float(w.w), inv) & 255u;
        const uint32_t packed = q0 | (q1 << 8) | (q2 << 16) | (q3 << 24);       // inv == 0 -> codes 0
        *(uint32_t*)(xq + (canonical ? k0 : plane_pos(k0, K))) = packed;
        if (tap_codes) *(uint32_t*)(tap_codes + k0) = packed;
        qs = dp4a_us(0x01010101u, (int)packed, qs);
    });
    qs = warp_sum_i(qs);
    if (x.lane == 0) atomicAdd(acc_qs(x) + par, qs);
    if (x.tid == 0) {
        scal(x)[0] = amax;
        acc_amax(x)[par ^ 1u] = 0u;        // last read behind the second barrier of the previous call
        acc_qs(x)[par ^ 1u] = 0;
    }
    if (pk >= 0) x.stamp(pl, pk + 2);
    __syncthreads();
    const int tot = acc_qs(x)[par];
    par ^= 1u;
    return tot;
}

// rstd and the activation scale s = (amax * rstd) / 127 (R13) from a sum of squares; ONE thread's arithmetic
__device__ __forceinline__ float act_scale(double ss, int K, float eps, float amax)
{
    const float ms = (float)(ss / (double)K);
    const float rstd = fdiv(1.0f, __fsqrt_rn(fadd(ms, eps)));
    return amax == 0.0f ? 0.0f : fdiv(fmul(amax, rstd), 127.0f);
}

// ONE warp, behind the barriers of absmax_quant: the activation scale of the vector whose amax is in scal[0], from the NWARPS
// warp sums of squares in red_d (any tree: DESIGN.md 5.3).  The embedding: every CTA holds the whole vector; U and G: the scale
// CTA gathered the workers' partial sums with the data (hop_gather) and the scale travels on as one word of the A / T part.
// Valid in lane 0.
template <class S>
__device__ __forceinline__ float scale_from_warps(const Ctx<S>& x, int K)
{
    double s = x.lane < NWARPS ? red_d(x)[x.lane] : 0.0;
#pragma unroll
    for (int o = NWARPS / 2; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    return act_scale(s, K, x.P.eps, scal(x)[0]);
}

// the elements a thread holds after gathering a slot-structured mailbox part (U or G): chunk ci = tid + j*THREADS is
// piece ci % pps of slot ci / pps; slot g carries elements starts[g] .. starts[g+1]-1
// DENSE: every slot is full and as long as its owner's element count: chunk ci holds the elements 4 ci .. 4 ci + 3
template <int NJ, bool DENSE>
struct SlotEnum {
    const uint4 (&v)[NJ];
    const int* starts;
    int tid, nslots, pps;
    template <typename F>
    __device__ __forceinline__ void operator()(F f) const
    {
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const int ci = tid + j * THREADS;
            if (ci < nslots * pps) {
                if (DENSE) {
                    f(4 * ci, v[j]);
                } else {
                    const int g = ci / pps, piece = ci - g * pps;
                    const int k0 = starts[g] + 4 * piece;
                    if (k0 < starts[g + 1]) f(k0, v[j]);
                }
            }
        }
    }
};

// ------------------------------------------------------------------------------------------------
// integer dot products
// ------------------------------------------------------------------------------------------------
// Sign dot products of up to NR rows against the plane-ordered codes in shared memory (S2 / S7) over the sign
// words [w0, w1) of each row: returns, in every lane, 128 * sum_{bit=1} q_k of row r in p[r] AFTER the caller
// reduces across lanes.  (dp4a of the mask 0x01010101 << i against plane i gives 2^i * partial sum.)
template <int NR>
__device__ __forceinline__ void sign_partial(const uint32_t* const (&rowp)[NR], int nrows, int w0, int w1, const uint8_t* xq, int K,
                                             int lane, int (&p)[NR])
{
    int a[NR][8];
#pragma unroll
    for (int r = 0; r < NR; ++r)
#pragma unroll
        for (int i = 0; i < 8; ++i) a[r][i] = 0;
    const uint8_t* xlo = xq;
    const uint8_t* xhi = xq + (K >> 1);
#pragma unroll 2
    for (int w = w0 + lane; w < w1; w += 32) {
        const int4 lo = *(const int4*)(xlo + 16 * w);
        const int4 hi = *(const int4*)(xhi + 16 * w);
#pragma unroll
        for (int r = 0; r < NR; ++r) {
            if (r < nrows) {
                const uint32_t b = rowp[r][w];
                a[r][0] = dp4a_us(b & 0x01010101u, lo.x, a[r][0]);
                a[r][1] = dp4a_us(b & 0x02020202u, lo.y, a[r][1]);
                a[r][2] = dp4a_us(b & 0x04040404u, lo.z, a[r][2]);
                a[r][3] = dp4a_us(b & 0x08080808u, lo.w, a[r][3]);
                a[r][4] = dp4a_us(b & 0x10101010u, hi.x, a[r][4]);
                a[r][5] = dp4a_us(b & 0x20202020u, hi.y, a[r][5]);
                a[r][6] = dp4a_us(b & 0x40404040u, hi.z, a[r][6]);
                a[r][7] = dp4a_us(b & 0x80808080u, hi.w, a[r][7]);
            }
        }
    }
#pragma unroll
    for (int r = 0; r < NR; ++r)       // a[r][i] = 2^i * S_i  ->  128 * sum_i S_i
        p[r] = (a[r][0] << 7) + (a[r][1] << 6) + (a[r][2] << 5) + (a[r][3] << 4) + (a[r][4] << 3) + (a[r][5] << 2) +
               (a[r][6] << 1) + a[r][7];
}

// reduction of 4 per-lane values: lane 8r ends up with the warp total of p[r] (one REDUX per value)
__device__ __forceinline__ int reduce4(const int (&p)[4], int lane)
{
    const int t0 = __reduce_add_sync(0xffffffffu, p[0]), t1 = __reduce_add_sync(0xffffffffu, p[1]);
    const int t2 = __reduce_add_sync(0xffffffffu, p[2]), t3 = __reduce_add_sync(0xffffffffu, p[3]);
    const int r = lane >> 3;
    return r == 0 ? t0 : r == 1 ? t1 : r == 2 ? t2 : t3;
}
// same for 2 values: lane 16r ends up with the warp total of p[r]
__device__ __forceinline__ int reduce2(const int (&p)[2], int lane)
{
    const int t0 = __reduce_add_sync(0xffffffffu, p[0]), t1 = __reduce_add_sync(0xffffffffu, p[1]);
    return (lane & 16) ? t1 : t0;
}

template <int NR> struct RowReduce;       // lane (32 / NR) * r ends up with the warp total of p[r]
template <> struct RowReduce<4> { static __device__ __forceinline__ int run(const int (&p)[4], int lane) { return reduce4(p, lane); } };
template <> struct RowReduce<2> { static __device__ __forceinline__ int run(const int (&p)[2], int lane) { return reduce2(p, lane); } };

// int8 x int8 dot of `nbytes` plane-permuted LoRA-down weights (fetched into the stage with the rest of the item)
// with the codes at the same positions
__device__ __forceinline__ int trow_dot(const uint8_t* row, int nbytes, const uint8_t* xq, int lane)
{
    const int nch = nbytes >> 4;
    int s = 0;
    for (int ch = lane; ch < nch; ch += 32) {
        const int4 a = *(const int4*)(row + 16 * ch);
        const int4 q = *(const int4*)(xq + 16 * ch);
        s = dp4a_ss(a.x, q.x, s); s = dp4a_ss(a.y, q.y, s); s = dp4a_ss(a.z, q.z, s); s = dp4a_ss(a.w, q.w, s);
    }
    return warp_sum_i(s);
}

// ------------------------------------------------------------------------------------------------
// weight / state pipeline
// ------------------------------------------------------------------------------------------------
// issue the bulk copies of pipeline item `item` into its ring stage (one thread)
template <class S>
__device__ __forceinline__ void issue_item(const Ctx<S>& x, int item, int v0, int v1)
{
    const Params& P = x.P;
    const int st = item % P.stages;
    uint8_t* stage = x.sm + P.s_ring + (size_t)st * P.stage_bytes;
    uint64_t* bar = (uint64_t*)(x.sm + P.s_mbar) + st;
    const uint64_t pol = policy_evict_first();
    if (item < P.L) {
        if (x.service()) {
            const int ts = x.c - x.NW() - 1;          // task index of this service CTA; -1: the scale CTA streams nothing
            mbar_expect_tx(bar, ts >= 0 ? P.schunk_bytes : 0u);
            if (ts >= 0) bulk_g2s_stream(stage, P.schunks + ((size_t)item * (x.NS() - 1) + ts) * P.schunk_bytes, P.schunk_bytes, bar, pol);
            return;
        }
        const int* chs = (const int*)(x.sm + P.s_chs);
        const int ch0 = chs[x.c], nch = chs[x.c + 1] - ch0;
        const uint32_t ssm_b = (uint32_t)nch * x.d_state() * 4, conv_b = (uint32_t)nch * 16, econv_b = (uint32_t)x.gs() * 32;
        mbar_expect_tx(bar, P.chunk_bytes + P.blk_bytes + ssm_b + conv_b + econv_b);
        bulk_g2s_stream(stage, P.chunks + ((size_t)item * x.NW() + x.c) * P.chunk_bytes, P.chunk_bytes, bar, pol);
        bulk_g2s(stage + P.st_blk, P.blocks + (size_t)item * P.blk_bytes, P.blk_bytes, bar);
        bulk_g2s(stage + P.st_econv, P.conv + (size_t)item * P.conv_lstride + (size_t)x.d_inner() * 4, econv_b, bar);
        if (nch > 0) {
            bulk_g2s_stream(stage + P.st_ssm, P.ssm + (size_t)item * P.ssm_lstride + (size_t)ch0 * x.d_state(), ssm_b, bar, pol);
            bulk_g2s(stage + P.st_conv, P.conv + (size_t)item * P.conv_lstride + (size_t)ch0 * 4, conv_b, bar);
        }
    } else {
        const int row0 = v0 + (item - P.L) * P.lm_rows_item;
        const int nrows = min(P.lm_rows_item, v1 - row0);
        const uint32_t bytes = (uint32_t)nrows * x.d_model();
        mbar_expect_tx(bar, bytes);
        bulk_g2s_stream(stage, P.emb + (size_t)row0 * x.d_model(), bytes, bar, pol);
    }
}

template <class S>
__device__ __forceinline__ void wait_item(const Ctx<S>& x, int item)
{
    const int st = item % x.P.stages;
    uint64_t* bar = (uint64_t*)(x.sm + x.P.s_mbar) + st;
    const uint32_t parity = (uint32_t)(item / x.P.stages) & 1u;
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > SPIN_LIMIT) { poll_fail(x); break; }
    }
}

// The stores of one CTA into a record.  publish and reset use the SAME thread -> address map.
//   slot (U / G): thread t < pps writes 16-byte piece t of its slot
template <class S, typename F>
__device__ __forceinline__ void slot_store(const Ctx<S>& x, uint32_t* rec, uint32_t part_off, int slot_w, F piece_value)
{
    const int pps = slot_w >> 2;
    for (int t = x.tid; t < pps; t += THREADS) x_st128(rec + part_off + (size_t)x.c * slot_w + 4 * t, piece_value(t));
}
//   the worker's fp64 partial of a slot part: the last thread (a warp that publishes no slot piece)
template <class S>
__device__ __forceinline__ void partial_store(const Ctx<S>& x, uint32_t* rec, uint32_t part_off, uint32_t lo, uint32_t hi)
{
    if (x.tid == THREADS - 1) x_st64(rec + part_off + 2 * (size_t)x.c, lo, hi);
}
//   word (A / T): the lanes of one warp write the word to the small mailboxes the workers poll
//   ncta = how many CTAs (0 .. ncta-1) poll the word: the workers, or everybody (0 = the workers)
template <class S>
__device__ __forceinline__ void word_store(const Ctx<S>& x, uint32_t* rec, uint32_t part_off, int idx, int M, uint32_t value, int ncta = 0)
{
    const Params& P = x.P;
    const int nm = mbox_count(ncta > 0 ? ncta : x.NW(), M);
    for (int m = x.lane; m < nm; m += 32) x_st32(rec + P.x_main + (size_t)m * P.x_small + part_off + idx, value);
}

// load time: replace A_log by A = -exp(A_log) inside every chunk (same sp_expf as the step would use; R10)
__global__ void k_mega_prepare(uint8_t* chunks, size_t n_chunks, uint32_t chunk_bytes, uint32_t c_alog, int nch_max)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_chunks * (size_t)nch_max) return;
    float* p = (float*)(chunks + (i / nch_max) * chunk_bytes + c_alog) + (i % nch_max);
    *p = -sp_expf(*p);
}

// every exchange word starts as "not written" (SENT); the words of a small mailbox that are never written (the pads that
// round the A and T parts up to whole 16-byte chunks: hop_gather tests whole chunks) hold 0 for good
__global__ void k_mega_init_x(uint32_t* xbuf, size_t n_records, uint32_t x_main, uint32_t x_small, uint32_t x_A, int n_A, uint32_t x_T,
                              int n_ttask, int i_sg, int i_slm)
{
    const size_t rec_words = (size_t)x_main + (size_t)MBOX * x_small;
    const size_t n = n_records * rec_words;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const size_t w = i % rec_words;
        uint32_t v = SENT;
        if (w >= x_main) {
            const uint32_t o = (uint32_t)((w - x_main) % x_small);
            const bool used = (o >= x_A && o < x_A + (uint32_t)n_A) || (o >= x_T && o < x_T + (uint32_t)n_ttask) || o == x_T + (uint32_t)i_sg ||
                              o == x_T + (uint32_t)i_slm;
            if (!used) v = 0u;
        }
        xbuf[i] = v;
    }
}

template <class S, bool TAPS, bool PROF>
__global__ void __launch_bounds__(THREADS, 1) k_mega(const Params P)
{
    extern __shared__ __align__(128) uint8_t sm[];
    __shared__ int s_dead;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, c = blockIdx.x;
    Ctx<S> x{ P, sm, tid, lane, wid, c, &s_dead, PROF && P.prof != nullptr };
    constexpr int NJ_G = Ctx<S>::NJG, NJ_U = Ctx<S>::NJU, NJ_0 = Ctx<S>::NJ0;

    int* chs = (int*)(sm + P.s_chs);
    int* ors = (int*)(sm + P.s_ors);
    uint64_t* mbar = (uint64_t*)(sm + P.s_mbar);
    uint8_t* xq = sm + P.s_xq;
    float* s_bc = (float*)(sm + P.s_bc);             // B' [gs] (fp32)
    double* s_cd = (double*)(sm + P.s_cd);           // C' [gs] as fp64: converted once, read by every channel of the state update
    float* s_u = (float*)(sm + P.s_u);
    float* s_z = (float*)(sm + P.s_z);
    float* s_x = (float*)(sm + P.s_x);
    float* s_dt = (float*)(sm + P.s_dt);
    double* s_vin = (double*)(sm + P.s_v);
    double* s_vout = s_vin + x.r_pad();
    int* s_eacc = (int*)(sm + P.s_eacc);
    int* s_acc_in = (int*)(sm + P.s_acc_in);
    int* s_acc_out = (int*)(sm + P.s_acc_out);
    const int NW = x.NW(), NS = x.NS();
    const bool service = c >= NW;
    const int sv = c - NW;                           // index among the service CTAs (if service): 0 = the scale CTA, 1 .. NS-1 hold row tasks
    const int ts = sv - 1, NT = NS - 1;              // task index / number of task CTAs

    for (int g = tid; g <= NW; g += THREADS) {
        chs[g] = own_start(g, x.d_inner(), NW);
        ors[g] = own_start(g, x.d_model(), NW);
    }
    if (tid < 2 * x.r_pad()) s_vin[tid] = 0.0;
    if (tid == 0) {
        s_dead = 0;
        for (int s = 0; s < P.stages; ++s) mbar_init(mbar + s, 1);
        fence_mbar_init();
    }
    __syncthreads();
    constexpr bool kEven = Ctx<S>::kEven;
    const int ch0 = service ? 0 : (kEven ? c * Ctx<S>::kNch : chs[c]), nch = service ? 0 : (kEven ? Ctx<S>::kNch : chs[c + 1] - ch0);
    const int or0 = service ? 0 : (kEven ? c * Ctx<S>::kNor : ors[c]), nor = service ? 0 : (kEven ? Ctx<S>::kNor : ors[c + 1] - or0);
    const int v0 = (int)(((long long)c * P.vocab) / x.G()), v1 = (int)(((long long)(c + 1) * P.vocab) / x.G());
    const int n_lm_items = (v1 - v0 + P.lm_rows_item - 1) / P.lm_rows_item;
    const int n_items = P.L + n_lm_items;
    if (tid == 0)
        for (int it = 0; it < P.stages && it < n_items; ++it) issue_item(x, it, v0, v1);

    const int ps = P.pos[0] & 3;                     // conv ring slot this step writes
    const int h0 = nch > 0 ? ch0 / x.headdim() : 0, h1 = nch > 0 ? (ch0 + nch - 1) / x.headdim() : -1;
    const bool taps_on = TAPS && P.taps != nullptr;
    const size_t rec_words = (size_t)P.x_main + (size_t)MBOX * P.x_small;
    auto mbox = [&](int M) { return (size_t)P.x_main + (size_t)mbox_of(c, M) * P.x_small; };      // offset of the small mailbox this worker polls
    const int rtid = THREADS - 1 - tid;              // the small gathers (A, T) are polled from the last warp down
    uint32_t* s_slotU = (uint32_t*)(sm + P.s_slot);
    uint32_t* s_slotG = s_slotU + x.u_slot();
    if (tid < x.u_slot() + x.g_slot()) s_slotU[tid] = 0u;      // pad words of the slots are published as 0
    // K-split of the out_proj sign rows: every (row pair, K part) is one warp task
    const int KS = (THREADS >= 1024 && x.Wout() >= 128) ? 4 : (x.Wout() >= 64 ? 2 : 1);
    const int tbytes = x.d_inner() / x.tsplit();         // bytes of one out_proj LoRA-down partial task
    // service: what this CTA holds of each dealt list
    const bool tasks = service && ts >= 0;
    const int n_sig = tasks ? dealt(x.n_bcdt(), ts, NT) : 0, n_lin = tasks ? dealt(x.r(), ts, NT) : 0,
              n_tt = tasks ? dealt(x.n_ttask(), ts, NT) : 0;

    // ---------------- S0 embedding + the first norm/quantise, redundantly in every CTA ----------------
    int qsum;
    unsigned par = 0u;                               // call parity of absmax_quant (its accumulators alternate)
    if (tid < 4) acc_amax(x)[tid] = 0u;              // acc_amax[2] | acc_qs[2]
    __syncthreads();
    {
        int tok = P.tokens[0];
        if (tok < 0 || tok >= P.vocab) {
            if (tid == 0 && c == 0) atomicOr(P.err, 1);
            tok = tok < 0 ? 0 : P.vocab - 1;
        }
        const int8_t* erow = P.emb + (size_t)tok * x.d_model();
        const float es = P.emb_s[tok];
        uint4 v[NJ_0];
        double ss = 0.0;
#pragma unroll
        for (int j = 0; j < NJ_0; ++j) {
            const int k0 = 4 * (tid + j * THREADS);
            if (k0 < x.d_model()) {
                uint32_t w[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float u = fmul(es, (float)erow[k0 + e]);
                    ss = dacc(ss, u, u);
                    w[e] = __float_as_uint(fmul(u, P.first_norm_w[k0 + e]));
                    if (k0 + e >= or0 && k0 + e < or0 + nor) s_u[k0 + e - or0] = u;
                }
                v[j] = make_uint4(w[0], w[1], w[2], w[3]);
            }
        }
        ss = warp_sum(ss);
        if (lane == 0) red_d(x)[wid] = ss;           // read by warp 0 behind the barriers of absmax_quant
        uint8_t* tp0 = (taps_on && c == 0 && P.L > 0) ? P.taps : nullptr;
        auto en = [&](auto f) {
#pragma unroll
            for (int j = 0; j < NJ_0; ++j) {
                const int k0 = 4 * (tid + j * THREADS);
                if (k0 < x.d_model()) f(k0, v[j]);
            }
        };
        qsum = absmax_quant(x, en, x.d_model(), P.L == 0, tp0 ? (int8_t*)(tp0 + P.tl.off[0]) : nullptr, par);
        if (wid == 0) {
            const float sc = scale_from_warps(x, x.d_model());
            if (lane == 0) scal(x)[1] = sc;          // scale of the layer-0 in_proj codes (L == 0: of the LM-head codes)
        }
        __syncthreads();
    }

    // =============================================== layers ===============================================
    for (int l = 0; l < P.L; ++l) {
        uint8_t* stage = sm + P.s_ring + (size_t)(l % P.stages) * P.stage_bytes;
        const uint8_t* blk = stage + P.st_blk;
        uint8_t* tp = taps_on ? P.taps + (size_t)l * P.tap_lstride : nullptr;
        float* conv_l = P.conv + (size_t)l * P.conv_lstride;
        uint32_t* rec = P.xbuf + ((size_t)P.set * P.L + l) * rec_words;                       // this step's record of layer l
        uint32_t* recc = P.xbuf + ((size_t)(P.set ^ 1u) * P.L + l) * rec_words;               // the next step's: own words are reset here
        DFSSM_STAMP(l, 0);
        if (x.prof && tid == 0) P.prof[((size_t)c * (P.L + 1) + l) * PROF_NPH + 31] = globaltimer_ns();
        wait_item(x, l);
        DFSSM_STAMP(l, 1);

        if (service) {
            // ================= service CTA: rows whose result every worker needs =================
            // ---- in_proj: B|C|dt sign rows and LoRA-down rows dealt to this CTA; raw int32 results are published ----
            {
                const uint32_t* bits = (const uint32_t*)(stage + P.sc_sign);
                for (int k0 = wid; k0 < n_sig + n_lin; k0 += NWARPS) {
                    // the LoRA-down rows go first (the workers need t_in before the accumulators of the B|C|dt rows)
                    const int k = k0 < n_lin ? n_sig + k0 : k0 - n_lin;
                    int val, idx;
                    if (k < n_sig) {
                        const uint32_t* const rowp[1] = { bits + (size_t)k * x.Win() };
                        int p[1];
                        sign_partial<1>(rowp, 1, 0, x.Win(), xq, x.d_model(), lane, p);
                        val = 2 * (warp_sum_i(p[0]) / 128) - qsum;       // exact: every term is a multiple of 128
                        idx = ts + k * NT;
                    } else {
                        const int kk = k - n_sig;
                        val = trow_dot(stage + P.sc_tin + (size_t)kk * x.d_model(), x.d_model(), xq, lane);
                        idx = x.n_bcdt() + ts + kk * NT;
                    }
                    word_store(x, rec, P.x_A, idx, M_A, (uint32_t)val ^ IBIAS);
                }
            }
            // ---- the scale CTA: the scale of the layer-0 in_proj codes (made with the embedding) travels with A; the later
            //      layers' scales are published as soon as their U has been gathered (end of the loop body) ----
            if (sv == 0 && wid == SCALE_WARP && l == 0) word_store(x, rec, P.x_A, x.n_early(), M_A, __float_as_uint(scal(x)[1]));
            DFSSM_STAMP(l, 2);
            x.gstamp(l, 29);
            // ---- gather G, codes of the whole gated vector ----
            int qsum_g;
            {
                uint4 vg[NJ_G];
                hop_gather<NJ_G>(x, rec + P.x_G, NW * x.g_slot() / 4, vg, tid, 0, sv == 0 ? rec + P.x_PG : nullptr);
                DFSSM_STAMP(l, 6);
                qsum_g = absmax_quant(x, SlotEnum<NJ_G, Ctx<S>::kDenseG>{ vg, chs, tid, NW, x.g_slot() >> 2 }, x.d_inner(), false, nullptr, par, l, 16);
            }
            if (sv == 0 && wid == SCALE_WARP) {     // the scale of the gated codes travels with T
                const float sc = scale_from_warps(x, x.d_inner());
                word_store(x, rec, P.x_T, x.i_sg(), M_T, __float_as_uint(sc));
            }
            (void)qsum_g;
            DFSSM_STAMP(l, 7);
            // ---- out_proj: LoRA-down partial tasks dealt to this CTA ----
            for (int k = wid; k < n_tt; k += NWARPS) {
                const int q = ts + k * NT, part = q % x.tsplit();
                const int t = trow_dot(stage + P.sc_tout + (size_t)k * tbytes, tbytes, xq + (size_t)part * tbytes, lane);
                word_store(x, rec, P.x_T, q, M_T, (uint32_t)t ^ IBIAS);
            }
            DFSSM_STAMP(l, 8);
            // ---- reset own words of the next step's record of this layer (this CTA is idle until U arrives) ----
            if (sv == 0 && wid == SCALE_WARP) {
                word_store(x, recc, P.x_A, x.n_early(), M_A, SENT);
                word_store(x, recc, P.x_T, x.i_sg(), M_T, SENT);
                if (l == P.L - 1) word_store(x, recc, P.x_T, x.i_slm(), M_T, SENT, GRID);
            }
            for (int k = wid; k < n_sig; k += NWARPS) word_store(x, recc, P.x_A, ts + k * NT, M_A, SENT);
            for (int k = wid; k < n_lin; k += NWARPS) word_store(x, recc, P.x_A, x.n_bcdt() + ts + k * NT, M_A, SENT);
            for (int k = wid; k < n_tt; k += NWARPS) word_store(x, recc, P.x_T, ts + k * NT, M_T, SENT);
            __syncthreads();                        // every thread is done with this stage's weights
            DFSSM_STAMP(l, 10);
        } else {
            // ================= worker CTA =================
            // ---- S2: z and x sign rows of this CTA (slots 0 .. 2 nch - 1: z rows, then x rows; the chunk pads them with zero rows
            //      to whole groups of NR_IN), NR_IN rows per warp pass, dealt from the top warp down ----
            {
                const uint32_t* bits = (const uint32_t*)(stage + P.c_in_bits);
                const int n_groups = (2 * nch + NR_IN - 1) / NR_IN;
                for (int q = NWARPS - 1 - wid; q < n_groups; q += NWARPS) {
                    const uint32_t* rowp[NR_IN];
#pragma unroll
                    for (int r = 0; r < NR_IN; ++r) rowp[r] = bits + (size_t)(NR_IN * q + r) * x.Win();
                    int p[NR_IN];
                    sign_partial<NR_IN>(rowp, NR_IN, 0, x.Win(), xq, x.d_model(), lane, p);
                    const int v = RowReduce<NR_IN>::run(p, lane);
                    if (lane % (32 / NR_IN) == 0) s_acc_in[NR_IN * q + lane / (32 / NR_IN)] = 2 * (v / 128) - qsum;
                }
            }
            DFSSM_STAMP(l, 2);
            x.gstamp(l, 30);
            // ---- gather A, first part: t_in and the scale (the chunks from word n_bcdt on; the task CTAs publish them first);
            //      v_j = a_s[j] * float(t_j).  The accumulators of the B|C|dt rows are polled word by word by the thread that
            //      finishes the row, behind its LoRA sum: they may arrive a whole epilogue later without anybody waiting ----
            const uint32_t* recA = rec + mbox(M_A) + P.x_A;
            {
                uint4 va[1];
                const int c0 = x.n_bcdt() / 4, nc1 = (x.n_A() + 3) / 4 - c0;
                hop_gather<1>(x, recA + 4 * c0, nc1, va, rtid);
                const float* a_s = (const float*)(blk + P.b_as_in);
                if (rtid < nc1) {
                    const int j = 0;
                    const int e0 = 4 * (c0 + rtid);
                    const uint32_t w[4] = { va[j].x, va[j].y, va[j].z, va[j].w };
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int e = e0 + i;
                        if (e == x.n_early()) {                   // scale of this layer's in_proj codes (made by service CTA 0)
                            scal(x)[1] = __uint_as_float(w[i]);
                            if (tp && c == 0) *(float*)(tp + P.tl.off[1]) = __uint_as_float(w[i]);
                        }
                        if (e >= x.n_bcdt() && e < x.n_early()) {
                            const int val = (int)(w[i] ^ IBIAS);
                            s_vin[e - x.n_bcdt()] = (double)fmul(a_s[e - x.n_bcdt()], (float)val);
                            if (tp && c == 0) ((int32_t*)(tp + P.tl.off[3]))[e - x.n_bcdt()] = val;
                        }
                    }
                }
            }
            __syncthreads();
            DFSSM_STAMP(l, 3);
            x.gstamp(l, 29);
            const float s_act = scal(x)[1];
            // ---- S3 stage 2 + S4 conv + dt softplus: own z|x rows and ALL B|C rows (+ own dt) ----
            {
                const int n_dt = (tp && c == 0) ? x.nheads() : (h1 - h0 + 1);
                float* ring = (float*)(stage + P.st_conv);
                const float* ering = (const float*)(stage + P.st_econv);
                // rows [first, first + count) of the index space (z | x | B|C | dt), skipping skip_len rows from skip_from on;
                // LP lanes share a row's LoRA sum; done by the threads [t0, t0 + nthr) (whole warps)
                auto epi = [&](auto lp_tag, int first, int count, int skip_from, int skip_len, int t0, int nthr) {
                  constexpr int LP = decltype(lp_tag)::value;
                  const int lt = tid - t0;
                  if (lt < 0 || lt >= nthr) return;
                  for (int ib = 0; ib < count; ib += nthr / LP) {          // warp-uniform trip count (shuffles inside)
                    int i = first + min(ib + lt / LP, count - 1);
                    if (i >= skip_from) i += skip_len;
                    const int sub = lt % LP;
                    const bool valid = ib + lt / LP < count;
                    int kind, slot = 0, e = 0;         // kind 0 z, 1 x, 2 B|C, 3 dt
                    if (i < nch) { kind = 0; slot = i; }
                    else if (i < 2 * nch) { kind = 1; slot = i; }
                    else if (i < 2 * nch + 2 * x.gs()) { kind = 2; e = i - 2 * nch; }
                    else { kind = 3; e = 2 * x.gs() + ((tp && c == 0) ? 0 : h0) + (i - 2 * nch - 2 * x.gs()); }
                    const bool own = kind < 2;
                    // LoRA-up row as 4-byte words: own rows are [slot][r_pad]; the B|C|dt rows of the shared block are stored word-major
                    // ([r_pad / 4][n_bcdt]) so that one thread per row reads shared memory without bank conflicts
                    const int* bw = own ? (const int*)(stage + P.c_in_B + (size_t)slot * x.r_pad()) : (const int*)(blk + P.b_eB) + e;
                    const int bstep = own ? 1 : x.n_bcdt();
                    // first look at the accumulator of a B|C|dt row BEFORE the LoRA sum: its trip to L2 runs under the sum; the spin
                    // behind the sum starts only if the word was not there yet (it is: the rows are published ~300 ns earlier)
                    uint32_t early = SENT;
                    if (!own && sub == 0 && valid) asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(early) : "l"(recA + e) : "memory");
                    double lo0 = 0.0, lo1 = 0.0;
                    for (int j4 = 4 * sub; j4 < x.r_pad(); j4 += 4 * LP) {         // pad entries of B are 0, pad entries of v are 0
                        const int w = bw[(j4 >> 2) * bstep];
                        const double2 v01 = *(const double2*)(s_vin + j4), v23 = *(const double2*)(s_vin + j4 + 2);
                        lo0 = __fma_rn((double)(int8_t)w, v01.x, lo0);
                        lo1 = __fma_rn((double)(int8_t)(w >> 8), v01.y, lo1);
                        lo0 = __fma_rn((double)(int8_t)(w >> 16), v23.x, lo0);
                        lo1 = __fma_rn((double)(w >> 24), v23.y, lo1);
                    }
                    lo0 += lo1;
#pragma unroll
                    for (int o = LP / 2; o > 0; o >>= 1) lo0 += __shfl_xor_sync(0xffffffffu, lo0, o);
                    if (sub != 0 || !valid) continue;
                    const float scale = own ? ((const float*)(stage + P.c_in_scale))[slot] : ((const float*)(blk + P.b_escale))[e];
                    const float bsv = own ? ((const float*)(stage + P.c_in_bs))[slot] : ((const float*)(blk + P.b_ebs))[e];
                    const int acc = own ? s_acc_in[slot] : (int)((early != SENT ? early : poll_word(x, recA + e)) ^ IBIAS);
                    const float lo = (float)lo0;
                    const float val = fmul(s_act, fadd(fmul(scale, (float)acc), fmul(bsv, lo)));
                    int row;                       // canonical in_proj row (for the taps)
                    bool tap_owner = true;
                    if (kind == 0) {
                        s_z[i] = siluf(val);           // the gate's factor
                        row = ch0 + i;
                    } else if (kind == 1) {
                        const int ic = i - nch;
                        float* rg = ring + 4 * ic;
                        const float s0 = rg[(ps + 1) & 3], s1 = rg[(ps + 2) & 3], s2 = rg[(ps + 3) & 3];
                        const float4 cw = *(const float4*)(stage + P.c_conv_w + 16 * ic);
                        float o = ((const float*)(stage + P.c_conv_b))[ic];
                        o = ffma(cw.x, s0, o); o = ffma(cw.y, s1, o); o = ffma(cw.z, s2, o); o = ffma(cw.w, val, o);
                        rg[ps] = val;
                        const float cv = siluf(o);
                        s_x[ic] = cv;
                        row = x.d_inner() + ch0 + ic;
                        if (tp) ((float*)(tp + P.tl.off[5]))[ch0 + ic] = cv;
                    } else if (kind == 2) {
                        const float* rg = ering + 4 * e;
                        const float s0 = rg[(ps + 1) & 3], s1 = rg[(ps + 2) & 3], s2 = rg[(ps + 3) & 3];
                        const float4 cw = *(const float4*)(blk + P.b_econv_w + 16 * e);
                        float o = ((const float*)(blk + P.b_econv_b))[e];
                        o = ffma(cw.x, s0, o); o = ffma(cw.y, s1, o); o = ffma(cw.z, s2, o); o = ffma(cw.w, val, o);
                        if (e % NW == c) conv_l[4 * (size_t)(x.d_inner() + e) + ps] = val;      // one worker keeps the state of this channel
                        const float cv = siluf(o);
                        if (e < x.gs()) s_bc[e] = cv;
                        else s_cd[e - x.gs()] = (double)cv;
                        row = 2 * x.d_inner() + e;
                        tap_owner = c == 0;
                        if (tp && tap_owner) ((float*)(tp + P.tl.off[5]))[x.d_inner() + e] = cv;
                    } else {
                        const int h = e - 2 * x.gs();
                        const float dtv = sp_softplusf(fadd(val, ((const float*)(blk + P.b_dtb))[h]));
                        s_dt[h] = dtv;
                        row = 2 * x.d_inner() + e;
                        tap_owner = c == 0;
                        if (tp && tap_owner) ((float*)(tp + P.tl.off[6]))[h] = dtv;
                    }
                    if (tp && tap_owner) {
                        ((float*)(tp + P.tl.off[4]))[row] = val;
                        ((int32_t*)(tp + P.tl.off[2]))[row] = acc;
                    }
                  }
                };
                // first half of the CTA: the 2 gs B|C rows, one thread per row (dense tails); second half, at the same time: the
                // few own rows (dt first: the longest tail; then x, z) with 4 lanes each if they fit one pass, else 2
                epi(std::integral_constant<int, LPB>{}, 2 * nch, 2 * x.gs(), 1 << 30, 0, 0, THREADS / 2);
                if constexpr (kEven && !TAPS) {          // the lane count is a compile-time choice: one copy of the epilogue code
                    constexpr int rows_own = 2 * Ctx<S>::kNch + (Ctx<S>::kNch + S::headdim - 1) / S::headdim + 1;
                    constexpr int LPO = 4 * rows_own <= THREADS / 2 ? 4 : 2;
                    epi(std::integral_constant<int, LPO>{}, 0, 2 * nch + n_dt, 2 * nch, 2 * x.gs(), THREADS / 2, THREADS / 2);
                } else if (4 * (2 * nch + n_dt) <= THREADS / 2)
                    epi(std::integral_constant<int, 4>{}, 0, 2 * nch + n_dt, 2 * nch, 2 * x.gs(), THREADS / 2, THREADS / 2);
                else
                    epi(std::integral_constant<int, 2>{}, 0, 2 * nch + n_dt, 2 * nch, 2 * x.gs(), THREADS / 2, THREADS / 2);
            }
            __syncthreads();
            DFSSM_STAMP(l, 4);

            // ---- S5 state update + readout, S6 gate: LPC lanes per channel; t = g*w is published as it is produced ----
            {
                double ss_own = 0.0;
                const int hpg = x.nheads() / x.ngroups();
                const float* Aneg = (const float*)(stage + P.c_alog);      // A = -exp(A_log), made by k_mega_prepare at load
                const float* Dv = (const float*)(stage + P.c_D);
                const float* gw = (const float*)(stage + P.c_gnorm);
                const int l16 = tid % LPC;
                for (int ib = 0; ib < nch; ib += THREADS / LPC) {        // warp-uniform trip count (shuffles inside)
                    const int i = min(ib + tid / LPC, nch - 1);
                    const bool valid = ib + tid / LPC < nch;
                    const int ch = ch0 + i, h = ch / x.headdim(), grp = h / hpg;
                    const float dtv = s_dt[h];
                    const float An = Aneg[i];
                    const float dA = sp_expf(fmul(dtv, An));
                    const float xv = s_x[i];
                    const float dtx = fmul(dtv, xv);
                    float* Hr = (float*)(stage + P.st_ssm) + (size_t)i * x.d_state();
                    const float* Bc = s_bc + grp * x.d_state();
                    const double* Cc = s_cd + grp * x.d_state();
                    double a0 = 0.0, a1 = 0.0;
                    for (int n4 = l16; valid && n4 < x.d_state() / 4; n4 += LPC) {
                        float4 hv = *(const float4*)(Hr + 4 * n4);
                        const float4 bv = *(const float4*)(Bc + 4 * n4);
                        const double2 c01 = *(const double2*)(Cc + 4 * n4), c23 = *(const double2*)(Cc + 4 * n4 + 2);
                        hv.x = ffma(dA, hv.x, fmul(dtx, bv.x));
                        hv.y = ffma(dA, hv.y, fmul(dtx, bv.y));
                        hv.z = ffma(dA, hv.z, fmul(dtx, bv.z));
                        hv.w = ffma(dA, hv.w, fmul(dtx, bv.w));
                        *(float4*)(Hr + 4 * n4) = hv;
                        a0 = __fma_rn(c01.x, (double)hv.x, a0); a1 = __fma_rn(c01.y, (double)hv.y, a1);
                        a0 = __fma_rn(c23.x, (double)hv.z, a0); a1 = __fma_rn(c23.y, (double)hv.w, a1);
                    }
                    double a = a0 + a1;
#pragma unroll
                    for (int o = LPC / 2; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o, LPC);
                    if (l16 == 0 && valid) {
                        a = dacc(a, Dv[i], xv);
                        const float y = (float)a;
                        const float gv = fmul(y, s_z[i]);
                        s_slotG[i] = __float_as_uint(fmul(gv, gw[i]));
                        ss_own = dacc(ss_own, gv, gv);
                        if (tp) { ((float*)(tp + P.tl.off[7]))[ch] = y; ((float*)(tp + P.tl.off[8]))[ch] = gv; }
                    }
                }
                x.stamp(l, 24);
                fence_proxy_async();               // the updated state is about to be read by the async proxy
                if (LPC < 32) ss_own = warp_sum_strided(ss_own, LPC);     // only the lanes 0, LPC, ... hold a value
                if (lane == 0) red_d(x)[wid] = ss_own;
                __syncthreads();
                x.stamp(l, 26);
                slot_store(x, rec, P.x_G, x.g_slot(), [&](int piece) { return *(const uint4*)(s_slotG + 4 * piece); });
                if (rtid == 0) {
                    double t4[4] = { 0.0, 0.0, 0.0, 0.0 };
#pragma unroll
                    for (int i = 0; i < NWARPS; ++i) t4[i & 3] += red_d(x)[i];
                    const double tot = (t4[0] + t4[1]) + (t4[2] + t4[3]);
                    partial_store(x, rec, P.x_PG, (uint32_t)__double2loint(tot), (uint32_t)__double2hiint(tot));
                }
                x.stamp(l, 27);
                if (tid == DMA_TID && nch > 0) {   // write the state slice back (async), while the exchange goes on
                    bulk_s2g_stream(P.ssm + (size_t)l * P.ssm_lstride + (size_t)ch0 * x.d_state(), stage + P.st_ssm, (uint32_t)nch * x.d_state() * 4,
                                    policy_evict_first());
                    bulk_s2g(conv_l + (size_t)ch0 * 4, stage + P.st_conv, (uint32_t)nch * 16);
                    bulk_commit();
                }
            }
            // reset own slots of the next step's record of this layer (same thread -> address map as the publishes), in the
            // shadow of the G exchange
            {
                slot_store(x, recc, P.x_U, x.u_slot(), [](int) { return make_uint4(SENT, SENT, SENT, SENT); });
                slot_store(x, recc, P.x_G, x.g_slot(), [](int) { return make_uint4(SENT, SENT, SENT, SENT); });
                partial_store(x, recc, P.x_PU, SENT, SENT);
                partial_store(x, recc, P.x_PG, SENT, SENT);
            }
            DFSSM_STAMP(l, 5);

            // ---- gather G, S6 absmax + quantise of the whole gated vector in every CTA ----
            int qsum_g;
            {
                uint4 vg[NJ_G];
                hop_gather<NJ_G>(x, rec + P.x_G, NW * x.g_slot() / 4, vg, tid, DFSSM_WG);
                DFSSM_STAMP(l, 6);
                qsum_g = absmax_quant(x, SlotEnum<NJ_G, Ctx<S>::kDenseG>{ vg, chs, tid, NW, x.g_slot() >> 2 }, x.d_inner(), false,
                                      (tp && c == 0) ? (int8_t*)(tp + P.tl.off[9]) : nullptr, par, l, 16);
            }
            DFSSM_STAMP(l, 7);
            // ---- S7: the out_proj sign rows ----
            {
                const uint32_t* bits = (const uint32_t*)(stage + P.c_out_bits);
                const int npair = (nor + 1) >> 1, wspan = x.Wout() / KS;
                for (int id = wid; id < npair * KS; id += NWARPS) {
                    const int pair = id / KS, half = id - pair * KS;
                    const int nrows = min(2, nor - 2 * pair);
                    const uint32_t* const rowp[2] = { bits + (size_t)(2 * pair) * x.Wout(), bits + (size_t)(2 * pair + (nrows > 1 ? 1 : 0)) * x.Wout() };
                    int p[2];
                    sign_partial<2>(rowp, nrows, half * wspan, half == KS - 1 ? x.Wout() : (half + 1) * wspan, xq, x.d_inner(), lane, p);
                    const int v = reduce2(p, lane);
                    const int r = lane >> 4;
                    if ((lane & 15) == 0 && r < nrows) s_acc_out[half * x.nor_max() + 2 * pair + r] = v;
                }
            }
            DFSSM_STAMP(l, 8);
            // ---- gather T: t_out = sum of the partial sums;  v_j = a_s[j] * float(t_j) ----
            {
                uint4 vt[1];
                hop_gather<1>(x, rec + mbox(M_T) + P.x_T, x.i_sg() / 4 + 1, vt, rtid);
                if (rtid == x.i_sg() / 4) {                   // scale of the gated codes (made by service CTA 0)
                    scal(x)[2] = __uint_as_float(vt[0].x);
                    if (tp && c == 0) *(float*)(tp + P.tl.off[10]) = __uint_as_float(vt[0].x);
                }
                if (rtid < x.i_sg() / 4) {
                    const float* a_s = (const float*)(blk + P.b_as_out);
                    const uint32_t w[4] = { vt[0].x, vt[0].y, vt[0].z, vt[0].w };
                    const int rows_per_chunk = 4 / x.tsplit();
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj) {
                        const int j = rtid * rows_per_chunk + jj;
                        if (jj < rows_per_chunk && j < x.r()) {
                            int t = 0;
                            for (int q = 0; q < x.tsplit(); ++q) t += (int)(w[jj * x.tsplit() + q] ^ IBIAS);
                            s_vout[j] = (double)fmul(a_s[j], (float)t);
                            if (tp && c == 0) ((int32_t*)(tp + P.tl.off[12]))[j] = t;
                        }
                    }
                }
            }
            __syncthreads();
            DFSSM_STAMP(l, 9);
            const float s_g = scal(x)[2];
            // ---- S7 epilogue + residual; t = u*w of the next norm is published as it is produced ----
            {
                double ss_u = 0.0;
                const int8_t* Bm = (const int8_t*)(stage + P.c_out_B);
                const float* scale = (const float*)(stage + P.c_out_scale);
                const float* bsv = (const float*)(stage + P.c_out_bs);
                const float* nw = (const float*)(stage + P.c_nnorm);
                for (int ib = 0; ib < nor; ib += THREADS / 4) {
                    const int i = ib + (tid >> 2), sub = tid & 3;
                    const bool valid = i < nor;
                    double lo = 0.0;
                    const int8_t* brow = Bm + (size_t)(valid ? i : 0) * x.r_pad();
                    if (valid)
                        for (int j = sub; j < x.r(); j += 4) lo = __fma_rn((double)brow[j], s_vout[j], lo);
                    lo += __shfl_xor_sync(0xffffffffu, lo, 1);
                    lo += __shfl_xor_sync(0xffffffffu, lo, 2);
                    if (sub != 0 || !valid) continue;
                    int p128 = s_acc_out[i];
                    for (int hh = 1; hh < KS; ++hh) p128 += s_acc_out[hh * x.nor_max() + i];
                    const int acc = 2 * (p128 / 128) - qsum_g;       // exact: every term is a multiple of 128
                    const float o = fmul(s_g, fadd(fmul(scale[i], (float)acc), fmul(bsv[i], (float)lo)));
                    const float un = fadd(s_u[i], o);
                    s_u[i] = un;
                    s_slotU[i] = __float_as_uint(fmul(un, nw[i]));
                    ss_u = dacc(ss_u, un, un);
                    if (tp) { ((float*)(tp + P.tl.off[13]))[or0 + i] = un; ((int32_t*)(tp + P.tl.off[11]))[or0 + i] = acc; }
                }
                ss_u = warp_sum_strided(ss_u, 4);           // only every fourth lane holds a value
                if (lane == 0) red_d(x)[wid] = ss_u;
                __syncthreads();                        // also: every thread is done with this stage's weights
                slot_store(x, rec, P.x_U, x.u_slot(), [&](int piece) { return *(const uint4*)(s_slotU + 4 * piece); });
                if (rtid == 0) {
                    double t4[4] = { 0.0, 0.0, 0.0, 0.0 };
#pragma unroll
                    for (int i = 0; i < NWARPS; ++i) t4[i & 3] += red_d(x)[i];
                    const double tot = (t4[0] + t4[1]) + (t4[2] + t4[3]);
                    partial_store(x, rec, P.x_PU, (uint32_t)__double2loint(tot), (uint32_t)__double2hiint(tot));
                }
            }
            DFSSM_STAMP(l, 10);
        }
        // ---- gather U, S1 of the next layer (or S8's norm) in every CTA ----
        {
            uint4 vu[NJ_U];
            hop_gather<NJ_U>(x, rec + P.x_U, NW * x.u_slot() / 4, vu, tid, service ? 0 : DFSSM_WU, (service && sv == 0) ? rec + P.x_PU : nullptr);
            DFSSM_STAMP(l, 11);
            x.gstamp(l, 28);
            uint8_t* tpn = (taps_on && c == 0 && l + 1 < P.L) ? P.taps + (size_t)(l + 1) * P.tap_lstride : nullptr;
            qsum = absmax_quant(x, SlotEnum<NJ_U, Ctx<S>::kDenseU>{ vu, ors, tid, NW, x.u_slot() >> 2 }, x.d_model(), l == P.L - 1,
                                tpn ? (int8_t*)(tpn + P.tl.off[0]) : nullptr, par, l, 20);
            // the scale of these codes is made by the scale CTA and travels with the next layer's A; the LM head gets it through T
            if (service && sv == 0 && wid == SCALE_WARP) {
                const float sc = scale_from_warps(x, x.d_model());
                if (l == P.L - 1) word_store(x, rec, P.x_T, x.i_slm(), M_T, __float_as_uint(sc), GRID);     // every CTA reads it
                else word_store(x, rec + rec_words, P.x_A, x.n_early(), M_A, __float_as_uint(sc));
            }
        }
        // ---- refill this layer's ring stage with the item `stages` ahead: after the gather, so that the bulk copies do
        //      not sit in front of its polls in the memory pipeline ----
        if (tid == DMA_TID) {
            bulk_wait_read0();                      // the state write-back has finished reading the stage
            if (l + P.stages < n_items) issue_item(x, l + P.stages, v0, v1);
        }
        DFSSM_STAMP(l, 12);
    }

    // =============================================== S8 LM head ===============================================
    if (P.L > 0 && tid == 0) {                       // scale of the final codes: word i_slm of the last layer's T part
        const uint32_t* w = P.xbuf + ((size_t)P.set * P.L + (P.L - 1)) * rec_words + P.x_main + (size_t)mbox_of(c, M_T) * P.x_small + P.x_T +
                            x.i_slm();
        uint32_t v, spins = 0;
        for (;;) {
            asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(w) : "memory");
            if (v != SENT) break;
            if (++spins > SPIN_LIMIT || *x.dead) { poll_fail(x); break; }
        }
        scal(x)[1] = __uint_as_float(v);
    }
    __syncthreads();
    const float s_act = scal(x)[1];
    for (int i = tid; i < nor; i += THREADS) P.u_out[or0 + i] = s_u[i];
    DFSSM_STAMP(P.L, 0);
    if (x.prof && tid == 0) P.prof[((size_t)c * (P.L + 1) + P.L) * PROF_NPH + 31] = globaltimer_ns();
    float best = -INFINITY;
    int besti = 0x7fffffff;
    for (int it = 0; it < n_lm_items; ++it) {
        const int item = P.L + it;
        wait_item(x, item);
        const uint8_t* stage = sm + P.s_ring + (size_t)(item % P.stages) * P.stage_bytes;
        const int row0 = v0 + it * P.lm_rows_item;
        const int nrows_it = min(P.lm_rows_item, v1 - row0);
        const int nchunk = x.d_model() >> 4;
        for (int q0 = 4 * wid; q0 < nrows_it; q0 += 4 * NWARPS) {
            const int nr = min(4, nrows_it - q0);
            int s[4] = { 0, 0, 0, 0 };
            for (int ch = lane; ch < nchunk; ch += 32) {
                const int4 q4 = *(const int4*)(xq + 16 * ch);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    if (r < nr) {
                        const int4 a4 = *(const int4*)(stage + (size_t)(q0 + r) * x.d_model() + 16 * ch);
                        s[r] = dp4a_ss(a4.x, q4.x, s[r]); s[r] = dp4a_ss(a4.y, q4.y, s[r]);
                        s[r] = dp4a_ss(a4.z, q4.z, s[r]); s[r] = dp4a_ss(a4.w, q4.w, s[r]);
                    }
                }
            }
            const int v = reduce4(s, lane);
            const int r = lane >> 3;
            if ((lane & 7) == 0 && r < nr) {
                const int row = row0 + q0 + r;
                const float lg = fmul((float)v, fmul(s_act, P.emb_s[row]));
                P.logits[row] = lg;
                if (lg > best || (lg == best && row < besti)) { best = lg; besti = row; }
            }
        }
        __syncthreads();
        if (tid == 0 && item + P.stages < n_items) issue_item(x, item + P.stages, v0, v1);
    }
    DFSSM_STAMP(P.L, 1);
    // ---- greedy token: CTA argmax -> global partials -> the last CTA to arrive finishes (lowest index on ties) ----
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, besti, o);
            if (ov > best || (ov == best && oi < besti)) { best = ov; besti = oi; }
        }
        float* rv = (float*)red_d(x);               // scratch: NWARPS floats | NWARPS ints
        int* ri = (int*)rv + NWARPS;
        __shared__ int s_last;
        if (lane == 0) { rv[wid] = best; ri[wid] = besti; }
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < NWARPS; ++w)
                if (rv[w] > best || (rv[w] == best && ri[w] < besti)) { best = rv[w]; besti = ri[w]; }
            P.am_val[c] = best;
            P.am_idx[c] = besti;
            __threadfence();
            const unsigned prev = atomicAdd(P.am_count, 1u);
            s_last = prev == (unsigned)x.G() - 1;
        }
        if (tid == DMA_TID) bulk_wait0();       // all state write-backs of this CTA are complete
        __syncthreads();
        if (s_last && wid == 0) {
            __threadfence();
            float b = -INFINITY;
            int bi = 0x7fffffff;
            for (int g = lane; g < x.G(); g += 32) {
                const float ov = __ldcg(P.am_val + g);
                const int oi = __ldcg(P.am_idx + g);
                if (ov > b || (ov == b && oi < bi)) { b = ov; bi = oi; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const float ov = __shfl_xor_sync(0xffffffffu, b, o);
                const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (ov > b || (ov == b && oi < bi)) { b = ov; bi = oi; }
            }
            if (lane == 0) {
                const int nx = bi == 0x7fffffff ? 0 : bi;
                P.next[0] = nx;
                P.tok_out[0] = nx;
                P.pos[0] = (ps + 1) & 3;
                *P.am_count = 0;
            }
        }
    }
}

}  // namespace mega
}  // namespace dfssm
