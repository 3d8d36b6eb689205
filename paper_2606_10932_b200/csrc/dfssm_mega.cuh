// "mega" path: the whole decode step of ONE sequence (S0, L x (S1..S7), S8) as ONE persistent
// cooperative kernel, one CTA per SM.  (the paper removes launch overhead with a CUDA graph;
// here the step is a single launch and the per-layer dependencies are resolved inside the kernel.)
//
// Design:
//   * Ownership.  CTA c owns d_inner channels [chs[c], chs[c+1]) -- their z and x in_proj rows, their conv
//     and SSM state, their gate -- and out_proj rows [ors[c], ors[c+1]) together with that slice of the
//     residual stream u (kept in shared memory for the whole step).  The B|C|dt in_proj rows and the
//     LoRA down-projection rows (t = A.xq) are "early tasks" dealt round-robin: task e belongs to CTA e % G.
//   * Weights.  dfssm_load_weights repacks every layer into one contiguous chunk per (layer, CTA)
//     (sign rows, LoRA-up rows, scales, conv taps, per-channel constants) plus one block per layer that
//     every CTA reads (the LoRA-up rows / scales / conv taps of the B|C|dt rows).  Chunk + block + the CTA's
//     slice of the SSM / conv state form one pipeline item, fetched by bulk async copies
//     (cp.async.bulk -> mbarrier) into a ring of shared-memory stages several layers AHEAD of the
//     dependency chain: addresses never depend on activations, so HBM stays busy while CTAs wait on
//     each other.  The LM head streams the int8 embedding through the same ring.
//   * Exchange.  Measured on B200: one store -> poll hop between CTAs through L2 costs >= ~0.9 us, so the
//     layer is built around FOUR all-gathers, two of them hidden behind sign-row work:
//       U : t_k = u_k * w_k (fp32) of the owned out rows + the CTA's partial sum of u^2 (fp64)
//           -> every CTA derives rstd / amax / the int8 codes of the WHOLE vector itself (S1)
//       A : raw int32 accumulators of the B|C|dt rows + t_in        (hidden behind the z|x sign rows)
//           -> every CTA finishes the B|C|dt epilogue, conv and softplus redundantly (S3, S4)
//       G : t_k = g_k * w_k (fp32) of the owned channels + partial sum of g^2  -> S6 everywhere
//       T : partial LoRA-down sums of out_proj                     (hidden behind the out_proj sign rows)
//     Buffers are self-validating ("Lamport" style): every 32-bit word is either the sentinel 0xffffffff
//     or payload (fp32 values are never that NaN; int32 values are stored with the sign bit flipped;
//     fp64 partials are 8-byte stores validated by their high word), so a hop is one store and one
//     successful poll, with no flag, fence or barrier.  A part can be PUSHED into M mailboxes (GRID / M CTAs poll each
//     copy).  Measured on the B200: U, G and A are fastest pulled from ONE copy; T, which every CTA
//     starts polling before it is written, is 2x faster pushed into 37 copies (polls delay stores to the same
//     lines).  The U / G payload of a CTA is one 128-byte slot written with 16-byte stores (a slot that straddles
//     a line costs ~1000 clocks per hop).  Records rotate over 4 (global layer counter mod 4): at layer l a CTA
//     resets its own slots of the record that layer l+2 will use (last used by layer l-2, which every CTA has
//     finished reading: it has since published for layer l-1), so the buffers stay L2-resident and a reset is at
//     least two hops old when the word is written or polled again.
//   * Arithmetic: identical to the chain path (dfssm_math.cuh; contract of DESIGN.md section 5).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "dfssm_kernels.cuh"
#include "dfssm_math.cuh"

namespace dfssm {
namespace mega {

constexpr int THREADS = 512;                  // 16 warps (measured: 32 warps only add issue pressure to the short phases)
constexpr int NWARPS = THREADS / 32;
constexpr int NJ_MAX = 3072 / THREADS;        // 16-byte chunks per thread when gathering U / G with run-time shapes (plan() checks)
constexpr int NJ_A = 1024 / THREADS;          // ... when gathering A
constexpr int NR_IN = THREADS >= 1024 ? 2 : 4;     // in_proj sign rows per warp pass
constexpr int LPR = THREADS / 512;            // lanes per row in the in_proj epilogue
constexpr int LPC = 16;                       // lanes per channel in the state update
constexpr int DMA_TID = 96;                   // the thread that issues the state write-back and the ring refills (a warp off the publish paths)
constexpr int KS_MAX = 4;                     // largest K-split of the out_proj sign rows
constexpr int MAX_STAGES = 8;
constexpr uint32_t SPIN_LIMIT = 1u << 20;     // ~0.3 s of polling, then the step aborts with an error flag
constexpr uint32_t SENT = 0xffffffffu;        // "not written yet"
constexpr uint32_t IBIAS = 0x80000000u;       // int32 payloads are stored xor IBIAS (|value| < 2^30)
constexpr int PROF_NPH = 32;                  // phase stamps per (CTA, layer) of the in-kernel profiler

struct Params {
    // ---- shape ----
    int L, d_model, d_inner, headdim, d_state, ngroups, nheads, r, vocab, n_bcdt, gs;
    float eps;
    int G;                       // grid size (CTAs), all co-resident
    int nch_max, nor_max, nb_max, n_slots, r_pad;
    int Win, Wout;               // sign words per row of in_proj / out_proj
    int n_early;                 // early tasks: n_bcdt sign rows + r LoRA-down rows
    int tsplit, n_ttask;         // out_proj LoRA-down rows are split into tsplit partial tasks each
    // ---- chunk layout (byte offsets inside one (layer, CTA) chunk) ----
    uint32_t c_in_bits, c_out_bits, c_in_B, c_out_B, c_in_scale, c_in_bs, c_out_scale, c_out_bs, c_conv_w, c_conv_b,
        c_alog, c_D, c_gnorm, c_nnorm, chunk_bytes;
    // ---- per-layer block read by every CTA (byte offsets) ----
    uint32_t b_eB, b_escale, b_ebs, b_econv_w, b_econv_b, b_dtb, b_as_in, b_as_out, blk_bytes;
    // ---- pipeline stage ----
    uint32_t st_blk, st_ssm, st_conv, st_econv, st_tin, st_tout, stage_bytes;
    int stages, lm_rows_item;
    // ---- exchange: M mailboxes x 4 rotating records; 32-bit word offsets inside one (record, mailbox) ----
    int M, gsz;                  // mailboxes, CTAs polling each (G = M * gsz); CTA c polls mailbox c / gsz
    int u_slot, u_dpos, g_slot, g_dpos;      // words per CTA slot of U / G, position of the fp64 partial inside it
    uint32_t x_U, x_A, x_G, x_T, x_words;
    // ---- shared memory carve ----
    uint32_t s_ring, s_mbar, s_xq, s_bc, s_u, s_z, s_x, s_dt, s_tq, s_v, s_eacc, s_acc_in, s_acc_out, s_chs, s_ors,
        s_part, s_red, s_slot, smem_bytes;
    // ---- device pointers ----
    const uint8_t* chunks;       // [L][G][chunk_bytes]
    const uint8_t* blocks;       // [L][blk_bytes]
    const int8_t* A_in;          // [L][r][d_model]  plane-permuted
    const int8_t* A_out;         // [L][r][d_inner]  plane-permuted
    float* ssm;                  // sequence 0 of layer 0; layer stride ssm_lstride floats
    float* conv;                 // [conv_dim][4] ring of sequence 0 of layer 0; layer stride conv_lstride floats
    size_t ssm_lstride, conv_lstride;
    const int8_t* emb; const float* emb_s; const float* first_norm_w;
    const int32_t* tokens; int32_t* next; int32_t* tok_out; int32_t* pos;
    float* logits; float* u_out;
    uint32_t* xbuf;              // [4 records][M][x_words]
    float* am_val; int* am_idx; unsigned* am_count;
    int* err;
    uint32_t rec0;               // record of layer 0 of this step (global layer counter mod 4)
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

// exchange words: relaxed gpu-scope accesses (served by L2; a 32-bit / 64-bit scalar access is single-copy atomic)
__device__ __forceinline__ void x_st32(uint32_t* p, uint32_t v)
{
    asm volatile("st.relaxed.gpu.global.b32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
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
struct ShapeRT { static constexpr bool kStatic = false; static constexpr int d_model = 0, d_inner = 0, headdim = 0, d_state = 0, ngroups = 0, r = 0; };
template <int DM, int DI, int HD, int DS, int NG, int R>
struct ShapeCT { static constexpr bool kStatic = true; static constexpr int d_model = DM, d_inner = DI, headdim = HD, d_state = DS, ngroups = NG, r = R; };

constexpr int GRID = 148;                       // one CTA per B200 SM
constexpr int MBOX = 37;                        // mailboxes allocated per record
// mailboxes actually used by each part (each must divide GRID and be <= MBOX): with M the payload is pushed M times and
// GRID / M CTAs poll each copy.  Tuned on the B200 (us per step, cfg 2): see DESIGN.md 6.2
#ifndef DFSSM_MU
#define DFSSM_MU 1
#define DFSSM_MG 1
#define DFSSM_MA 1
#define DFSSM_MT 37
#endif
// clocks a CTA waits after publishing G / U before its first poll: polls that reach a line before the data delay the
// stores to it (measured: 0 -> 0.501 ms/step, 300..700 -> 0.488)
#ifndef DFSSM_WG
#define DFSSM_WG 500
#define DFSSM_WU 500
#endif
constexpr int M_U = DFSSM_MU, M_G = DFSSM_MG, M_A = DFSSM_MA, M_T = DFSSM_MT;

// Ownership: CTA g owns elements [own_start(g, n), own_start(g + 1, n)) of a vector of length n (n % 4 == 0), in
// groups of 4 so that a gathered 16-byte chunk is four consecutive elements of one 16-element half block of codes.
__host__ __device__ constexpr int own_start(int g, int n) { return 4 * (int)(((long long)g * (n / 4)) / GRID); }
__host__ __device__ constexpr int own_max(int n) { return 4 * ((n / 4 + GRID - 1) / GRID); }
// words of one CTA's slot in a U / G mailbox: a power of two (16, 32, 64 ...), so that a slot never straddles a 128-byte
// line (measured: 80-byte slots cost ~1000 clocks per hop more than 64- or 128-byte ones)
__host__ __device__ constexpr int slot_words(int need) { int w = 4; while (w < need) w *= 2; return w; }
// 16-byte chunks per thread needed to gather the slots of a vector of length n (or to hold n / 4 chunks: n_flat)
__host__ __device__ constexpr int nj_slots(int n) { return (GRID * slot_words((own_max(n) + 1) / 2 * 2 + 2) / 4 + THREADS - 1) / THREADS; }

template <class S>
struct Ctx {
    const Params& P;
    uint8_t* sm;
    int tid, lane, wid, c;
    volatile int* dead;          // shared flag: a poll timed out -> stop spinning everywhere
    bool prof;                   // in-kernel profiler on (a compile-time false in the production instantiations)
    static constexpr int NJG = S::kStatic ? nj_slots(S::d_inner) : NJ_MAX;     // chunks per thread: gather G, gather U, embedding
    static constexpr int NJU = S::kStatic ? nj_slots(S::d_model) : NJ_MAX;
    static constexpr int NJ0 = S::kStatic ? (S::d_model / 4 + THREADS - 1) / THREADS : 8192 / 4 / THREADS;
#define DFSSM_DIM(n_) __device__ __forceinline__ int n_() const { return S::kStatic ? S::n_ : P.n_; }
    DFSSM_DIM(d_model) DFSSM_DIM(d_inner) DFSSM_DIM(headdim) DFSSM_DIM(d_state) DFSSM_DIM(ngroups) DFSSM_DIM(r)
#undef DFSSM_DIM
    __device__ __forceinline__ void stamp(int l, int k) const
    {
        if (prof && tid == 0) P.prof[((size_t)c * (P.L + 1) + l) * PROF_NPH + k] = clock64();
    }
    __device__ __forceinline__ constexpr int G() const { return GRID; }
    __device__ __forceinline__ constexpr int M() const { return MBOX; }
    __device__ __forceinline__ constexpr int gsz() const { return GRID / MBOX; }
    __device__ __forceinline__ int nheads() const { return d_inner() / headdim(); }
    __device__ __forceinline__ int gs() const { return ngroups() * d_state(); }
    __device__ __forceinline__ int n_bcdt() const { return 2 * gs() + nheads(); }
    __device__ __forceinline__ int nch_max() const { return own_max(d_inner()); }
    __device__ __forceinline__ int nor_max() const { return own_max(d_model()); }
    __device__ __forceinline__ int nb_max() const { return (n_bcdt() + GRID - 1) / GRID; }
    __device__ __forceinline__ int n_slots() const { return 2 * nch_max() + nb_max(); }
    __device__ __forceinline__ int r_pad() const { return (r() + 3) / 4 * 4; }
    __device__ __forceinline__ int Win() const { return d_model() / 32; }
    __device__ __forceinline__ int Wout() const { return d_inner() / 32; }
    __device__ __forceinline__ int n_early() const { return n_bcdt() + r(); }
    __device__ __forceinline__ int tsplit() const { return (d_inner() % 64 == 0 && 4 * r() <= GRID) ? 4 : (2 * r() <= GRID ? 2 : 1); }
    __device__ __forceinline__ int n_ttask() const { return r() * tsplit(); }
    // early task e = c + k G of this CTA that is a LoRA-down row (at most one: r <= G), or -1
    __device__ __forceinline__ int t_in_task() const
    {
        const int k = c >= n_bcdt() ? 0 : (n_bcdt() - c + GRID - 1) / GRID;
        const int e = c + k * GRID;
        return e < n_early() ? e : -1;
    }
    __device__ __forceinline__ int u_dpos() const { return (nor_max() + 1) / 2 * 2; }
    __device__ __forceinline__ int u_slot() const { return slot_words(u_dpos() + 2); }
    __device__ __forceinline__ int g_dpos() const { return (nch_max() + 1) / 2 * 2; }
    __device__ __forceinline__ int g_slot() const { return slot_words(g_dpos() + 2); }
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
    atomicExch(x.P.err, 2);
}

// ------------------------------------------------------------------------------------------------
// exchange: gather a self-validating buffer
// ------------------------------------------------------------------------------------------------
// Thread t owns the 16-byte chunks t, t + THREADS, ... (at most NJ) of the nw 32-bit words at buf.  Words
// behind nw count as valid.  If slot_w > 0 the buffer is a sequence of slots of slot_w words whose word dpos is
// the low half of an fp64 (any bit pattern: exempt; its high half at dpos + 1 validates it).
// Spins until every owned word has been written; the raw words come back in v[].  tix = the thread's index for
// the chunk ownership (tid, or reversed so that the small gathers are polled by the warps that have nothing else to do).
template <int NJ, class S>
__device__ __forceinline__ void hop_gather(const Ctx<S>& x, const uint32_t* buf, int nw, int slot_w, int dpos, uint4 (&v)[NJ], int tix, int first_wait = 0)
{
    if (first_wait > 0) {                          // polls that arrive before the data delay the stores to the same lines
        const long long t0 = clock64();
        while (clock64() - t0 < first_wait) {}
    }
    const int nchunk = (nw + 3) >> 2;
    bool need[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) need[j] = tix + j * THREADS < nchunk;
    uint32_t spins = 0;
    for (;;) {
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (need[j]) v[j] = x_ld128(buf + 4 * (tix + j * THREADS));
        bool all = true;
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (need[j]) {
                const int base = 4 * (tix + j * THREADS);
                const int ex = slot_w > 0 ? dpos - base % slot_w : -1;      // index of the exempt word inside this chunk
                const bool ok = (v[j].x != SENT || ex == 0) && (base + 1 >= nw || v[j].y != SENT) &&
                                (base + 2 >= nw || v[j].z != SENT || ex == 2) && (base + 3 >= nw || v[j].w != SENT);
                need[j] = !ok;
                all = all && ok;
            }
        if (all) break;
        if (++spins > SPIN_LIMIT || *x.dead) { poll_fail(x); break; }
    }
}

// scratch inside s_red: NWARPS floats (warp maxima) | NWARPS ints (warp code sums) | NWARPS doubles (warp sums)
template <class S>
__device__ __forceinline__ float* red_f(const Ctx<S>& x) { return (float*)(x.sm + x.P.s_red); }
template <class S>
__device__ __forceinline__ int* red_i(const Ctx<S>& x) { return (int*)(x.sm + x.P.s_red) + NWARPS; }
template <class S>
__device__ __forceinline__ double* red_d(const Ctx<S>& x) { return (double*)(x.sm + x.P.s_red + 8 * NWARPS); }

// S1 / S6 / S8 norm + quantise of a whole vector in every CTA.  `en(f)` calls f(k, bits) for every element this
// thread holds: bits = fp32 t_k = value_k * w_k;  ss_local = the partial sums of squares this thread holds (the
// per-CTA partials it gathered, or its own elements' squares for the embedding).  Every warp reduces the 16 warp
// results and derives rstd / amax / scale itself; every thread then quantises its elements.  Writes the codes to
// xq (plane order unless `canonical`), returns the sum of the codes and the activation scale s.
// Two __syncthreads.
template <class S, typename Enum>
__device__ __forceinline__ int norm_quant(const Ctx<S>& x, Enum en, double ss_local, int dstride, int dlane, int K, bool canonical, float& s_out,
                                          int8_t* tap_codes, int pl = 0, int pk = -1)
{
    const Params& P = x.P;
    uint8_t* xq = x.sm + P.s_xq;
    float* bc = (float*)(x.sm + P.s_part);
    float am = 0.0f;
    en([&](int, uint4 w) {
        am = fmaxf(fmaxf(am, fabsf(__uint_as_float(w.x))), fabsf(__uint_as_float(w.y)));
        am = fmaxf(fmaxf(am, fabsf(__uint_as_float(w.z))), fabsf(__uint_as_float(w.w)));
    });
    am = warp_max(am);
    ss_local = warp_sum_strided(ss_local, dstride);      // only the lanes dlane + k * dstride hold partial sums
    if (x.lane == 0) red_f(x)[x.wid] = am;
    if (x.lane == dlane) red_d(x)[x.wid] = ss_local;
    if (pk >= 0) x.stamp(pl, pk);
    __syncthreads();
    if (pk >= 0) x.stamp(pl, pk + 1);
    // every warp derives the constants itself from the NWARPS warp results (cheaper than a second barrier)
    static_assert(NWARPS == 16, "the reductions below read 16 warp results");
    float amax;
    double ss;
    {
        const float4* rf = (const float4*)red_f(x);
        const float4 a0 = rf[0], a1 = rf[1], a2 = rf[2], a3 = rf[3];
        amax = fmaxf(fmaxf(fmaxf(fmaxf(a0.x, a0.y), fmaxf(a0.z, a0.w)), fmaxf(fmaxf(a1.x, a1.y), fmaxf(a1.z, a1.w))),
                     fmaxf(fmaxf(fmaxf(a2.x, a2.y), fmaxf(a2.z, a2.w)), fmaxf(fmaxf(a3.x, a3.y), fmaxf(a3.z, a3.w))));
        const double2* rd = (const double2*)red_d(x);
        double2 d[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) d[i] = rd[i];
        ss = (((d[0].x + d[0].y) + (d[1].x + d[1].y)) + ((d[2].x + d[2].y) + (d[3].x + d[3].y))) +
             (((d[4].x + d[4].y) + (d[5].x + d[5].y)) + ((d[6].x + d[6].y) + (d[7].x + d[7].y)));
    }
    const float ms = (float)(ss / (double)K);
    const float rstd = fdiv(1.0f, __fsqrt_rn(fadd(ms, P.eps)));
    const float inv = amax == 0.0f ? 0.0f : fdiv(127.0f, amax);
    s_out = amax == 0.0f ? 0.0f : fdiv(fmul(amax, rstd), 127.0f);
    if (pk >= 0) x.stamp(pl, pk + 2);
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
    if (x.lane == 0) red_i(x)[x.wid] = qs;
    if (pk >= 0) x.stamp(pl, pk + 3);
    __syncthreads();
    const int4* ri = (const int4*)red_i(x);
    const int4 q0 = ri[0], q1 = ri[1], q2 = ri[2], q3 = ri[3];
    return ((q0.x + q0.y) + (q0.z + q0.w)) + ((q1.x + q1.y) + (q1.z + q1.w)) + ((q2.x + q2.y) + (q2.z + q2.w)) + ((q3.x + q3.y) + (q3.z + q3.w));
}

// the elements a thread holds after gathering a slot-structured mailbox part (U or G): chunk ci = tid + j*THREADS is
// piece ci % pps of slot ci / pps; slot g carries elements starts[g] .. starts[g+1]-1 and its fp64 partial at dpos
template <int NJ>
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
                const int g = ci / pps, piece = ci - g * pps;
                const int k0 = starts[g] + 4 * piece;
                if (k0 < starts[g + 1]) f(k0, v[j]);
            }
        }
    }
};
// sum of the fp64 partials found in this thread's gathered chunks
template <int NJ, class S>
__device__ __forceinline__ double slot_partials(const Ctx<S>& x, const uint4 (&v)[NJ], int nslots, int slot_w, int dpos)
{
    const int pps = slot_w >> 2;
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        const int ci = x.tid + j * THREADS;
        if (ci < nslots * pps) {
            const int g = ci / pps, ex = dpos - 4 * (ci - g * pps);
            if (ex == 0) s += __hiloint2double((int)v[j].y, (int)v[j].x);
            else if (ex == 2) s += __hiloint2double((int)v[j].w, (int)v[j].z);
        }
    }
    return s;
}

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
        const int* chs = (const int*)(x.sm + P.s_chs);
        const int ch0 = chs[x.c], nch = chs[x.c + 1] - ch0;
        const uint32_t ssm_b = (uint32_t)nch * x.d_state() * 4, conv_b = (uint32_t)nch * 16, econv_b = (uint32_t)x.gs() * 32;
        const int e_t = x.t_in_task();                                      // LoRA-down row of in_proj this CTA owns (or -1)
        const uint32_t tin_b = e_t >= 0 ? (uint32_t)x.d_model() : 0u;
        const uint32_t tout_b = x.c < x.n_ttask() ? (uint32_t)(x.d_inner() / x.tsplit()) : 0u;
        mbar_expect_tx(bar, P.chunk_bytes + P.blk_bytes + ssm_b + conv_b + econv_b + tin_b + tout_b);
        if (tin_b) bulk_g2s_stream(stage + P.st_tin, P.A_in + ((size_t)item * x.r() + (e_t - x.n_bcdt())) * x.d_model(), tin_b, bar, pol);
        if (tout_b)
            bulk_g2s_stream(stage + P.st_tout, P.A_out + ((size_t)item * x.r() + x.c / x.tsplit()) * x.d_inner() + (size_t)(x.c % x.tsplit()) * tout_b, tout_b, bar, pol);
        bulk_g2s_stream(stage, P.chunks + ((size_t)item * x.G() + x.c) * P.chunk_bytes, P.chunk_bytes, bar, pol);
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

// The stores of one CTA into the M mailboxes of a record.  publish and reset use the SAME thread -> address map, so
// a reset and the later publish of a word are ordered by program order of one thread.
//   slot (U / G): thread t < M * pps writes 16-byte piece t % pps of its slot in mailbox t / pps
template <class S, typename F>
__device__ __forceinline__ void slot_store(const Ctx<S>& x, uint32_t* rec, uint32_t part_off, int slot_w, int M, F piece_value)
{
    const Params& P = x.P;
    const int pps = slot_w >> 2;
    for (int t = x.tid; t < M * pps; t += THREADS) {
        const int m = t / pps, piece = t - m * pps;
        x_st128(rec + (size_t)m * P.x_words + part_off + (size_t)x.c * slot_w + 4 * piece, piece_value(piece));
    }
}
//   word (A / T): the lanes of one warp write the word to all mailboxes
template <class S>
__device__ __forceinline__ void word_store(const Ctx<S>& x, uint32_t* rec, uint32_t part_off, int idx, int M, uint32_t value)
{
    const Params& P = x.P;
    for (int m = x.lane; m < M; m += 32) x_st32(rec + (size_t)m * P.x_words + part_off + idx, value);
}

// load time: replace A_log by A = -exp(A_log) inside every chunk (same sp_expf as the step would use; R10)
__global__ void k_mega_prepare(uint8_t* chunks, size_t n_chunks, uint32_t chunk_bytes, uint32_t c_alog, int nch_max)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_chunks * (size_t)nch_max) return;
    float* p = (float*)(chunks + (i / nch_max) * chunk_bytes + c_alog) + (i % nch_max);
    *p = -sp_expf(*p);
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
    float* s_bc = (float*)(sm + P.s_bc);
    float* s_u = (float*)(sm + P.s_u);
    float* s_z = (float*)(sm + P.s_z);
    float* s_x = (float*)(sm + P.s_x);
    float* s_dt = (float*)(sm + P.s_dt);
    double* s_vin = (double*)(sm + P.s_v);
    double* s_vout = s_vin + x.r_pad();
    int* s_eacc = (int*)(sm + P.s_eacc);
    int* s_acc_in = (int*)(sm + P.s_acc_in);
    int* s_acc_out = (int*)(sm + P.s_acc_out);

    for (int g = tid; g <= x.G(); g += THREADS) {
        chs[g] = own_start(g, x.d_inner());
        ors[g] = own_start(g, x.d_model());
    }
    if (tid < 2 * x.r_pad()) s_vin[tid] = 0.0;
    if (tid == 0) {
        s_dead = 0;
        for (int s = 0; s < P.stages; ++s) mbar_init(mbar + s, 1);
        fence_mbar_init();
    }
    __syncthreads();
    const int ch0 = chs[c], nch = chs[c + 1] - ch0;
    const int or0 = ors[c], nor = ors[c + 1] - or0;
    const int v0 = (int)(((long long)c * P.vocab) / x.G()), v1 = (int)(((long long)(c + 1) * P.vocab) / x.G());
    const int n_lm_items = (v1 - v0 + P.lm_rows_item - 1) / P.lm_rows_item;
    const int n_items = P.L + n_lm_items;
    if (tid == 0)
        for (int it = 0; it < P.stages && it < n_items; ++it) issue_item(x, it, v0, v1);

    const int ps = P.pos[0] & 3;                     // conv ring slot this step writes
    const int nb_tasks = c < x.n_early() ? (x.n_early() - c + x.G() - 1) / x.G() : 0;      // early tasks of this CTA
    const int h0 = nch > 0 ? ch0 / x.headdim() : 0, h1 = nch > 0 ? (ch0 + nch - 1) / x.headdim() : -1;
    const bool taps_on = TAPS && P.taps != nullptr;
    const size_t rec_words = (size_t)x.M() * P.x_words;
    auto mbox = [&](int M) { return (size_t)(c / (GRID / M)) * P.x_words; };      // offset of the mailbox this CTA polls of a part pushed M times
    const int rtid = THREADS - 1 - tid;              // the small gathers (A, T) are polled from the last warp down
    uint32_t* s_slotU = (uint32_t*)(sm + P.s_slot);
    uint32_t* s_slotG = s_slotU + x.u_slot();
    if (tid < x.u_slot() + x.g_slot()) s_slotU[tid] = 0u;      // pad words of the slots are published as 0
    // K-split of the out_proj sign rows: every (row pair, K part) is one warp task
    const int KS = (THREADS >= 1024 && x.Wout() >= 128) ? 4 : (x.Wout() >= 64 ? 2 : 1);
    const int tbytes = x.d_inner() / x.tsplit();         // bytes of one out_proj LoRA-down partial task

    // ---------------- S0 embedding + the first norm/quantise, redundantly in every CTA ----------------
    float s_act;                                     // scale of the current activation codes
    int qsum;
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
        uint8_t* tp0 = (taps_on && c == 0 && P.L > 0) ? P.taps : nullptr;
        auto en = [&](auto f) {
#pragma unroll
            for (int j = 0; j < NJ_0; ++j) {
                const int k0 = 4 * (tid + j * THREADS);
                if (k0 < x.d_model()) f(k0, v[j]);
            }
        };
        qsum = norm_quant(x, en, ss, 1, 0, x.d_model(), P.L == 0, s_act, tp0 ? (int8_t*)(tp0 + P.tl.off[0]) : nullptr);
        if (tp0 && tid == 0) *(float*)(tp0 + P.tl.off[1]) = s_act;
    }

    // =============================================== layers ===============================================
    for (int l = 0; l < P.L; ++l) {
        uint8_t* stage = sm + P.s_ring + (size_t)(l % P.stages) * P.stage_bytes;
        const uint8_t* blk = stage + P.st_blk;
        uint8_t* tp = taps_on ? P.taps + (size_t)l * P.tap_lstride : nullptr;
        float* conv_l = P.conv + (size_t)l * P.conv_lstride;
        uint32_t* rec = P.xbuf + (size_t)((P.rec0 + (uint32_t)l) & 3u) * rec_words;          // published into (all mailboxes)
        uint32_t* recc = P.xbuf + (size_t)((P.rec0 + (uint32_t)l + 2u) & 3u) * rec_words;     // reset for layer l + 2
        DFSSM_STAMP(l, 0);
        if (x.prof && tid == 0) P.prof[((size_t)c * (P.L + 1) + l) * PROF_NPH + 31] = globaltimer_ns();
        wait_item(x, l);
        DFSSM_STAMP(l, 1);
        // ---- early tasks: B|C|dt sign rows and LoRA-down rows of this CTA; raw int32 results are published ----
        {
            const uint32_t* bits = (const uint32_t*)(stage + P.c_in_bits);
            for (int k = wid; k < nb_tasks; k += NWARPS) {
                const int e = c + k * x.G();
                int val;
                if (e < x.n_bcdt()) {
                    const uint32_t* const rowp[1] = { bits + (size_t)(2 * x.nch_max() + k) * x.Win() };
                    int p[1];
                    sign_partial<1>(rowp, 1, 0, x.Win(), xq, x.d_model(), lane, p);
                    val = 2 * (warp_sum_i(p[0]) / 128) - qsum;       // exact: every term is a multiple of 128
                } else {
                    val = trow_dot(stage + P.st_tin, x.d_model(), xq, lane);
                }
                word_store(x, rec, P.x_A, e, M_A, (uint32_t)val ^ IBIAS);
                if (lane == 0 && tp && e >= x.n_bcdt()) ((int32_t*)(tp + P.tl.off[3]))[e - x.n_bcdt()] = val;
            }
        }
        // ---- S2: z and x sign rows of this CTA, NR_IN rows per warp pass, dealt from the top warp down ----
        {
            const uint32_t* bits = (const uint32_t*)(stage + P.c_in_bits);
            const int n_tasks = 2 * nch;
            for (int q = NWARPS - 1 - wid; NR_IN * q < n_tasks; q += NWARPS) {
                const uint32_t* rowp[NR_IN];
                int slot[NR_IN];
                const int nrows = min(NR_IN, n_tasks - NR_IN * q);
#pragma unroll
                for (int r = 0; r < NR_IN; ++r) {
                    const int t = NR_IN * q + r;
                    slot[r] = r < nrows ? (t < nch ? t : x.nch_max() + (t - nch)) : 0;
                    rowp[r] = bits + (size_t)slot[r] * x.Win();
                }
                int p[NR_IN];
                sign_partial<NR_IN>(rowp, nrows, 0, x.Win(), xq, x.d_model(), lane, p);
                const int v = RowReduce<NR_IN>::run(p, lane);
                const int r = lane / (32 / NR_IN);
                if (lane % (32 / NR_IN) == 0 && r < nrows) s_acc_in[slot[r]] = 2 * (v / 128) - qsum;
            }
        }
        DFSSM_STAMP(l, 2);
        {   // reset own slots of the record two layers ahead (same thread -> address map as the publishes); the warps
            // that do it are not the ones polling A, so this costs nothing on the critical path
            slot_store(x, recc, P.x_U, x.u_slot(), M_U, [](int) { return make_uint4(SENT, SENT, SENT, SENT); });
            slot_store(x, recc, P.x_G, x.g_slot(), M_G, [](int) { return make_uint4(SENT, SENT, SENT, SENT); });
            for (int k = wid; k < nb_tasks; k += NWARPS) word_store(x, recc, P.x_A, c + k * x.G(), M_A, SENT);
            if (wid == 0 && c < x.n_ttask()) word_store(x, recc, P.x_T, c, M_T, SENT);
        }

        // ---- gather A: accumulators of all B|C|dt rows and t_in;  v_j = a_s[j] * float(t_j) ----
        {
            uint4 va[NJ_A];
            hop_gather<NJ_A>(x, rec + mbox(M_A) + P.x_A, x.n_early(), 0, 0, va, rtid);
            const float* a_s = (const float*)(blk + P.b_as_in);
#pragma unroll
            for (int j = 0; j < NJ_A; ++j) {
                const int e0 = 4 * (rtid + j * THREADS);
                const uint32_t w[4] = { va[j].x, va[j].y, va[j].z, va[j].w };
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int e = e0 + i;
                    if (e < x.n_early()) {
                        const int val = (int)(w[i] ^ IBIAS);
                        if (e < x.n_bcdt()) s_eacc[e] = val;
                        else s_vin[e - x.n_bcdt()] = (double)fmul(a_s[e - x.n_bcdt()], (float)val);
                    }
                }
            }
        }
        __syncthreads();
        DFSSM_STAMP(l, 3);
        // ---- S3 stage 2 + S4 conv + dt softplus: LPR lanes per row; own z|x rows and ALL B|C rows (+ own dt) ----
        {
            const int n_dt = tp ? x.nheads() : (h1 - h0 + 1);
            const int n_rows = 2 * nch + 2 * x.gs() + n_dt;
            float* ring = (float*)(stage + P.st_conv);
            const float* ering = (const float*)(stage + P.st_econv);
            // rows [first, first + count) of the index space (z | x | B|C | dt), skipping skip_len rows from skip_from on;
            // LP lanes share a row's LoRA sum
            // done by the threads [t0, t0 + nthr) (whole warps)
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
                else if (i < 2 * nch) { kind = 1; slot = x.nch_max() + (i - nch); }
                else if (i < 2 * nch + 2 * x.gs()) { kind = 2; e = i - 2 * nch; }
                else { kind = 3; e = 2 * x.gs() + (tp ? 0 : h0) + (i - 2 * nch - 2 * x.gs()); }
                const bool own = kind < 2;
                // LoRA-up row as 4-byte words: own rows are [slot][r_pad]; the B|C|dt rows of the shared block are stored word-major
                // ([r_pad / 4][n_bcdt]) so that one thread per row reads shared memory without bank conflicts
                const int* bw = own ? (const int*)(stage + P.c_in_B + (size_t)slot * x.r_pad()) : (const int*)(blk + P.b_eB) + e;
                const int bstep = own ? 1 : x.n_bcdt();
                double lo0 = 0.0, lo1 = 0.0;
                for (int j4 = 4 * sub; j4 < x.r_pad(); j4 += 4 * LP) {         // pad entries of B are 0, pad entries of v are 0
                    const int w = bw[(j4 >> 2) * bstep];
                    lo0 = __fma_rn((double)(int8_t)w, s_vin[j4], lo0);
                    lo1 = __fma_rn((double)(int8_t)(w >> 8), s_vin[j4 + 1], lo1);
                    lo0 = __fma_rn((double)(int8_t)(w >> 16), s_vin[j4 + 2], lo0);
                    lo1 = __fma_rn((double)(w >> 24), s_vin[j4 + 3], lo1);
                }
                lo0 += lo1;
#pragma unroll
                for (int o = LP / 2; o > 0; o >>= 1) lo0 += __shfl_xor_sync(0xffffffffu, lo0, o);
                if (sub != 0 || !valid) continue;
                const float scale = own ? ((const float*)(stage + P.c_in_scale))[slot] : ((const float*)(blk + P.b_escale))[e];
                const float bsv = own ? ((const float*)(stage + P.c_in_bs))[slot] : ((const float*)(blk + P.b_ebs))[e];
                const int acc = own ? s_acc_in[slot] : s_eacc[e];
                const float lo = (float)lo0;
                const float val = fmul(s_act, fadd(fmul(scale, (float)acc), fmul(bsv, lo)));
                int row;                       // canonical in_proj row (for the taps)
                bool tap_owner = true;
                if (kind == 0) {
                    s_z[i] = val;
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
                    tap_owner = e % x.G() == c;
                    if (tap_owner) conv_l[4 * (size_t)(x.d_inner() + e) + ps] = val;      // the early-task owner keeps the state
                    const float cv = siluf(o);
                    s_bc[e] = cv;
                    row = 2 * x.d_inner() + e;
                    if (tp && tap_owner) ((float*)(tp + P.tl.off[5]))[x.d_inner() + e] = cv;
                } else {
                    const int h = e - 2 * x.gs();
                    const float dtv = sp_softplusf(fadd(val, ((const float*)(blk + P.b_dtb))[h]));
                    s_dt[h] = dtv;
                    row = 2 * x.d_inner() + e;
                    tap_owner = e % x.G() == c;
                    if (tp && tap_owner) ((float*)(tp + P.tl.off[6]))[h] = dtv;
                }
                if (tp && tap_owner) {
                    ((float*)(tp + P.tl.off[4]))[row] = val;
                    ((int32_t*)(tp + P.tl.off[2]))[row] = acc;
                }
              }
            };
            // first half of the CTA: the 2 gs B|C rows, one thread per row (dense tails); second half, at the same time: the
            // few own rows (z, x, dt) with 4 lanes each
            epi(std::integral_constant<int, 1>{}, 2 * nch, 2 * x.gs(), 1 << 30, 0, 0, THREADS / 2);
            epi(std::integral_constant<int, 4>{}, 0, 2 * nch + n_dt, 2 * nch, 2 * x.gs(), THREADS / 2, THREADS / 2);
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
                const float sz = siluf(s_z[i]);             // all lanes: free in SIMT, and off the tail of the reduction
                float* Hr = (float*)(stage + P.st_ssm) + (size_t)i * x.d_state();
                const float* Bc = s_bc + grp * x.d_state();
                const float* Cc = s_bc + x.gs() + grp * x.d_state();
                double a = 0.0;
                for (int n4 = l16; valid && n4 < x.d_state() / 4; n4 += LPC) {
                    float4 hv = *(const float4*)(Hr + 4 * n4);
                    const float4 bv = *(const float4*)(Bc + 4 * n4);
                    const float4 cv = *(const float4*)(Cc + 4 * n4);
                    hv.x = ffma(dA, hv.x, fmul(dtx, bv.x));
                    hv.y = ffma(dA, hv.y, fmul(dtx, bv.y));
                    hv.z = ffma(dA, hv.z, fmul(dtx, bv.z));
                    hv.w = ffma(dA, hv.w, fmul(dtx, bv.w));
                    *(float4*)(Hr + 4 * n4) = hv;
                    a = dacc(a, cv.x, hv.x); a = dacc(a, cv.y, hv.y); a = dacc(a, cv.z, hv.z); a = dacc(a, cv.w, hv.w);
                }
#pragma unroll
                for (int o = LPC / 2; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o, LPC);
                if (l16 == 0 && valid) {
                    a = dacc(a, Dv[i], xv);
                    const float y = (float)a;
                    const float gv = fmul(y, sz);
                    s_slotG[i] = __float_as_uint(fmul(gv, gw[i]));
                    ss_own = dacc(ss_own, gv, gv);
                    if (tp) { ((float*)(tp + P.tl.off[7]))[ch] = y; ((float*)(tp + P.tl.off[8]))[ch] = gv; }
                }
            }
            x.stamp(l, 24);
            fence_proxy_async();               // the updated state is about to be read by the async proxy
            x.stamp(l, 25);
            ss_own = warp_sum_strided(ss_own, LPC);     // only lanes 0 and 16 hold a value
            if (lane == 0) red_d(x)[wid] = ss_own;
            __syncthreads();
            x.stamp(l, 26);
            slot_store(x, rec, P.x_G, x.g_slot(), M_G, [&](int piece) {
                uint4 w = *(const uint4*)(s_slotG + 4 * piece);
                const int ex = x.g_dpos() - 4 * piece;
                if (ex == 0 || ex == 2) {
                    double t4[4] = { 0.0, 0.0, 0.0, 0.0 };
#pragma unroll
                    for (int i = 0; i < NWARPS; ++i) t4[i & 3] += red_d(x)[i];
                    const double tot = (t4[0] + t4[1]) + (t4[2] + t4[3]);
                    const uint32_t lo = (uint32_t)__double2loint(tot), hi = (uint32_t)__double2hiint(tot);
                    if (ex == 0) { w.x = lo; w.y = hi; } else { w.z = lo; w.w = hi; }
                }
                return w;
            });
            x.stamp(l, 27);
            if (tid == DMA_TID && nch > 0) {   // write the state slice back (async), while the exchange goes on
                bulk_s2g_stream(P.ssm + (size_t)l * P.ssm_lstride + (size_t)ch0 * x.d_state(), stage + P.st_ssm, (uint32_t)nch * x.d_state() * 4,
                                policy_evict_first());
                bulk_s2g(conv_l + (size_t)ch0 * 4, stage + P.st_conv, (uint32_t)nch * 16);
                bulk_commit();
            }
        }
        DFSSM_STAMP(l, 5);

        // ---- gather G, S6 norm + quantise of the whole gated vector in every CTA ----
        float s_g;
        int qsum_g;
        {
            uint4 vg[NJ_G];
            hop_gather<NJ_G>(x, rec + mbox(M_G) + P.x_G, x.G() * x.g_slot(), x.g_slot(), x.g_dpos(), vg, tid, DFSSM_WG);
            DFSSM_STAMP(l, 6);
            const double ssl = slot_partials<NJ_G>(x, vg, x.G(), x.g_slot(), x.g_dpos());
            const int gpps = x.g_slot() >> 2;            // the fp64 partials sit in the lanes (g_dpos / 4) mod pps
            qsum_g = norm_quant(x, SlotEnum<NJ_G>{ vg, chs, tid, x.G(), gpps }, ssl, gpps < 32 ? gpps : 1, gpps < 32 ? (x.g_dpos() >> 2) % gpps : 0,
                                x.d_inner(), false, s_g,
                                (tp && c == 0) ? (int8_t*)(tp + P.tl.off[9]) : nullptr, l, 16);
            if (tp && c == 0 && tid == 0) *(float*)(tp + P.tl.off[10]) = s_g;
        }
        DFSSM_STAMP(l, 7);
        // ---- S7: LoRA-down partial task (warp 0, published) and the out_proj sign rows (other warps) ----
        if (wid == 0) {
            if (c < x.n_ttask()) {
                const int part = c % x.tsplit();
                const int t = trow_dot(stage + P.st_tout, tbytes, xq + (size_t)part * tbytes, lane);
                word_store(x, rec, P.x_T, c, M_T, (uint32_t)t ^ IBIAS);
            }
        } else {
            const uint32_t* bits = (const uint32_t*)(stage + P.c_out_bits);
            const int npair = (nor + 1) >> 1, wspan = x.Wout() / KS;
            for (int id = wid - 1; id < npair * KS; id += NWARPS - 1) {
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
            hop_gather<1>(x, rec + mbox(M_T) + P.x_T, x.n_ttask(), 0, 0, vt, rtid);
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
        __syncthreads();
        DFSSM_STAMP(l, 9);
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
            slot_store(x, rec, P.x_U, x.u_slot(), M_U, [&](int piece) {
                uint4 w = *(const uint4*)(s_slotU + 4 * piece);
                const int ex = x.u_dpos() - 4 * piece;
                if (ex == 0 || ex == 2) {
                    double t4[4] = { 0.0, 0.0, 0.0, 0.0 };
#pragma unroll
                    for (int i = 0; i < NWARPS; ++i) t4[i & 3] += red_d(x)[i];
                    const double tot = (t4[0] + t4[1]) + (t4[2] + t4[3]);
                    const uint32_t lo = (uint32_t)__double2loint(tot), hi = (uint32_t)__double2hiint(tot);
                    if (ex == 0) { w.x = lo; w.y = hi; } else { w.z = lo; w.w = hi; }
                }
                return w;
            });
        }
        DFSSM_STAMP(l, 10);
        // ---- gather U, S1 of the next layer (or S8's norm) in every CTA ----
        {
            uint4 vu[NJ_U];
            hop_gather<NJ_U>(x, rec + mbox(M_U) + P.x_U, x.G() * x.u_slot(), x.u_slot(), x.u_dpos(), vu, tid, DFSSM_WU);
            DFSSM_STAMP(l, 11);
            const double ssl = slot_partials<NJ_U>(x, vu, x.G(), x.u_slot(), x.u_dpos());
            uint8_t* tpn = (taps_on && c == 0 && l + 1 < P.L) ? P.taps + (size_t)(l + 1) * P.tap_lstride : nullptr;
            const int upps = x.u_slot() >> 2;
            qsum = norm_quant(x, SlotEnum<NJ_U>{ vu, ors, tid, x.G(), upps }, ssl, upps < 32 ? upps : 1, upps < 32 ? (x.u_dpos() >> 2) % upps : 0,
                              x.d_model(), l == P.L - 1, s_act,
                              tpn ? (int8_t*)(tpn + P.tl.off[0]) : nullptr, l, 20);
            if (tpn && tid == 0) *(float*)(tpn + P.tl.off[1]) = s_act;
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
        float* rv = red_f(x);
        int* ri = red_i(x);
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
