// "mega" path: the whole decode step of ONE sequence (S0, L x (S1..S7), S8) as ONE persistent
// cooperative kernel, one CTA per SM.  (the paper removes launch overhead with a CUDA graph;
// here the step is a single launch and the per-layer dependencies are resolved inside the kernel.)
//
// Design:
//   * Ownership.  CTA c owns d_inner channels [chs[c], chs[c+1]) -- their z and x in_proj rows, their conv
//     and SSM state, their gate -- and out_proj rows [ors[c], ors[c+1]) together with that slice of the
//     residual stream u (kept in shared memory for the whole step).  The B|C|dt in_proj rows and the
//     LoRA down-projection rows (t = A.xq) are dealt round-robin: row e belongs to CTA e % G.
//   * Weights.  dfssm_load_weights repacks every layer into one contiguous chunk per (layer, CTA)
//     (sign rows, LoRA-up rows, scales, conv taps, per-channel constants).  A chunk plus the CTA's slice
//     of the SSM / conv state is one pipeline item, fetched by bulk async copies (cp.async.bulk ->
//     mbarrier) into a ring of shared-memory stages several layers AHEAD of the dependency chain:
//     addresses never depend on activations, so HBM stays busy while CTAs wait on each other.
//     The LM head streams the int8 embedding through the same ring.
//   * Exchange.  All-gathers between CTAs use flag-in-data 64-bit words in global memory (L2):
//     {payload32, flag32} or {7 int8 codes, flag8}, written with st.relaxed.gpu.b64 and polled with
//     ld.relaxed.gpu.b64 -- a 64-bit scalar access is single-copy atomic, so a matching flag proves the
//     payload; no fence, no separate barrier, one L2 round trip per hop.  Flags are unique per use.
//     Per layer: stats(u) -> codes(u) -> t_in -> B'|C'|dt -> stats(g) -> codes(g) -> t_out.
//   * Arithmetic: identical to the chain path (dfssm_math.cuh; contract of DESIGN.md section 5).
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "dfssm_kernels.cuh"
#include "dfssm_math.cuh"

namespace dfssm {
namespace mega {

constexpr int THREADS = 512;
constexpr int NWARPS = THREADS / 32;
constexpr int MAX_STAGES = 8;
constexpr uint32_t SPIN_LIMIT = 1u << 21;     // ~0.5 s of polling, then the step aborts with an error flag
constexpr int CODES_PER_WORD = 7;
constexpr int PROF_NPH = 16;                  // phase stamps per (CTA, layer) of the in-kernel profiler

struct Params {
    // ---- shape ----
    int L, d_model, d_inner, headdim, d_state, ngroups, nheads, r, vocab, n_bcdt, gs;
    float eps;
    int G;                       // grid size (CTAs), all co-resident
    int nch_max, nor_max, nb_max, n_slots, r_pad;
    int Win, Wout;               // sign words per row of in_proj / out_proj
    int wpc1, wpc3;              // code words per CTA in the u / g code exchanges
    // ---- chunk layout (byte offsets inside one (layer, CTA) chunk) ----
    uint32_t c_in_bits, c_out_bits, c_in_B, c_out_B, c_in_scale, c_in_bs, c_out_scale, c_out_bs, c_conv_w, c_conv_b,
        c_e_conv_w, c_e_conv_b, c_e_dtb, c_alog, c_D, c_gnorm, c_nnorm, c_as_in, c_as_out, chunk_bytes;
    // ---- pipeline stage ----
    uint32_t st_ssm, st_conv, stage_bytes;
    int stages, lm_rows_item;
    // ---- shared memory carve ----
    uint32_t s_ring, s_mbar, s_xq, s_bc, s_u, s_z, s_x, s_tq, s_vin, s_vout, s_acc_in, s_acc_out, s_chs, s_ors,
        s_stats, s_red, smem_bytes;
    // ---- device pointers ----
    const uint8_t* chunks;       // [L][G][chunk_bytes]
    const int8_t* A_in;          // [L][r][d_model]  plane-permuted
    const int8_t* A_out;         // [L][r][d_inner]  plane-permuted
    float* ssm;                  // sequence 0 of layer 0; layer stride ssm_lstride floats
    float* conv;                 // [conv_dim][4] ring of sequence 0 of layer 0; layer stride conv_lstride floats
    size_t ssm_lstride, conv_lstride;
    const int8_t* emb; const float* emb_s; const float* first_norm_w;
    const int32_t* tokens; int32_t* next; int32_t* tok_out; int32_t* pos;
    float* logits; float* u_out;
    uint64_t *x_stat1, *x_code1, *x_t, *x_bc, *x_stat3, *x_code3, *x_t4;
    float* am_val; int* am_idx; unsigned* am_count;
    int* err;
    uint32_t base32, e255;
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
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src_smem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void ll_store(uint64_t* p, uint64_t v)
{
    asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint64_t ll_load(const uint64_t* p)
{
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint64_t ll_pack32(uint32_t payload, uint32_t flag) { return ((uint64_t)flag << 32) | payload; }

__device__ __forceinline__ int4 ldg_nc16(const void* p)
{
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// position of canonical element k inside a plane-ordered code vector of length K: word w = k/32, in-word
// p = 8j + i; planes 0..3 live in the first half (16 B per word), planes 4..7 in the second half.
__device__ __forceinline__ int plane_pos(int k, int K)
{
    const int w = k >> 5, p = k & 31, j = p >> 3, i = p & 7;
    return (i < 4 ? 0 : (K >> 1)) + 16 * w + 4 * (i & 3) + j;
}

struct Ctx {
    const Params& P;
    uint8_t* sm;
    int tid, lane, wid, c;
    volatile int* dead;          // shared flag: a poll timed out -> stop spinning everywhere
};

__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
// in-kernel profiler: thread 0 of every CTA stamps its SM clock at phase k of layer l
#define DFSSM_STAMP(l_, k_)                                                                            \
    do {                                                                                               \
        if (P.prof && tid == 0) P.prof[((size_t)c * (P.L + 1) + (l_)) * PROF_NPH + (k_)] = clock64();  \
    } while (0)

__device__ __forceinline__ void poll_fail(const Ctx& x)
{
    *x.dead = 1;
    atomicExch(x.P.err, 2);
}

// Poll n flag-in-data words; consume(idx, word) is called once per word by the thread that polled it.
// Each thread keeps up to 4 loads in flight.  flag is compared with the top `fbits` bits (32 or 8).
template <int FBITS, typename F>
__device__ __forceinline__ void poll_words(const Ctx& x, const uint64_t* buf, int n, uint32_t flag, F consume)
{
    for (int base = x.tid; base < n; base += THREADS * 4) {
        uint64_t v[4];
        bool ok[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) ok[j] = (base + j * THREADS) >= n;
        uint32_t spins = 0;
        for (;;) {
            bool all = true;
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (!ok[j]) v[j] = ll_load(buf + base + j * THREADS);
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (!ok[j]) {
                    ok[j] = (uint32_t)(v[j] >> (64 - FBITS)) == flag;
                    all = all && ok[j];
                }
            if (all) break;
            if (++spins > SPIN_LIMIT || *x.dead) { poll_fail(x); break; }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (base + j * THREADS < n) consume(base + j * THREADS, v[j]);
    }
}

// block-wide (sum of doubles, max of floats); result to every thread.  Two __syncthreads.
__device__ __forceinline__ void block_sum_max(const Ctx& x, double& s, float& m)
{
    double* rd = (double*)(x.sm + x.P.s_red);             // [NWARPS]
    float* rf = (float*)(rd + NWARPS);                    // [NWARPS]
    s = warp_sum(s);
    m = warp_max(m);
    if (x.lane == 0) { rd[x.wid] = s; rf[x.wid] = m; }
    __syncthreads();
    double s2 = 0.0;
    float m2 = 0.0f;
#pragma unroll
    for (int i = 0; i < NWARPS; ++i) { s2 += rd[i]; m2 = fmaxf(m2, rf[i]); }
    __syncthreads();
    s = s2;
    m = m2;
}

// quantiser constants from (sum of squares, amax) of a vector of length d (R4, R13)
__device__ __forceinline__ void quant_consts(double ss, float amax, int d, float eps, float& inv, float& s)
{
    const float ms = (float)(ss / (double)d);
    const float rstd = fdiv(1.0f, __fsqrt_rn(fadd(ms, eps)));
    inv = amax == 0.0f ? 0.0f : fdiv(127.0f, amax);
    s = amax == 0.0f ? 0.0f : fdiv(fmul(amax, rstd), 127.0f);
}

// Sign dot products of up to 4 rows against the plane-ordered codes in shared memory (S2 / S7):
// returns in lane 8*r the value sum_k sign_rk * q_k of row r.  rowp[r] points at the row's packed words.
__device__ __forceinline__ int sign_dot4(const uint32_t* (&rowp)[4], int nrows, int W, const uint8_t* xq, int K,
                                         int qsum, int lane)
{
    int a[4][8];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < 8; ++i) a[r][i] = 0;
    const uint8_t* xlo = xq;
    const uint8_t* xhi = xq + (K >> 1);
    for (int w = lane; w < W; w += 32) {
        const int4 lo = *(const int4*)(xlo + 16 * w);
        const int4 hi = *(const int4*)(xhi + 16 * w);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
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
    int p[4];
#pragma unroll
    for (int r = 0; r < 4; ++r)       // a[r][i] = 2^i * S_i  ->  128 * sum_i S_i
        p[r] = (a[r][0] << 7) + (a[r][1] << 6) + (a[r][2] << 5) + (a[r][3] << 4) + (a[r][4] << 3) + (a[r][5] << 2) +
               (a[r][6] << 1) + a[r][7];
    // transposing reduction: 4 values x 32 lanes -> lane 8r holds the total of row r
    const bool up16 = (lane & 16) != 0, up8 = (lane & 8) != 0;
    int k0 = up16 ? p[2] : p[0], k1 = up16 ? p[3] : p[1];
    int s0 = up16 ? p[0] : p[2], s1 = up16 ? p[1] : p[3];
    k0 += __shfl_xor_sync(0xffffffffu, s0, 16);
    k1 += __shfl_xor_sync(0xffffffffu, s1, 16);
    int v = up8 ? k1 : k0;
    const int sv = up8 ? k0 : k1;
    v += __shfl_xor_sync(0xffffffffu, sv, 8);
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    return 2 * (v / 128) - qsum;      // exact: every term is a multiple of 128
}

// int8 x int8 dot of a plane-permuted LoRA-down row (global memory) with the codes in shared memory.
// pre[] holds the row's first 8*32 16-byte chunks, loaded earlier so their latency is off the critical path.
constexpr int T_PRE = 8;
__device__ __forceinline__ void trow_prefetch(const int8_t* row, int K, int lane, int4 (&pre)[T_PRE])
{
    const int nch = K >> 4;
#pragma unroll
    for (int i = 0; i < T_PRE; ++i) {
        const int ch = lane + 32 * i;
        if (ch < nch) pre[i] = ldg_nc16(row + 16 * ch);
    }
}
__device__ __forceinline__ int trow_dot(const int8_t* row, int K, const uint8_t* xq, int lane, const int4 (&pre)[T_PRE])
{
    const int nch = K >> 4;
    int s = 0;
#pragma unroll
    for (int i = 0; i < T_PRE; ++i) {
        const int ch = lane + 32 * i;
        if (ch < nch) {
            const int4 q = *(const int4*)(xq + 16 * ch);
            s = dp4a_ss(pre[i].x, q.x, s); s = dp4a_ss(pre[i].y, q.y, s);
            s = dp4a_ss(pre[i].z, q.z, s); s = dp4a_ss(pre[i].w, q.w, s);
        }
    }
    for (int ch = lane + 32 * T_PRE; ch < nch; ch += 32) {
        const int4 a = ldg_nc16(row + 16 * ch);
        const int4 q = *(const int4*)(xq + 16 * ch);
        s = dp4a_ss(a.x, q.x, s); s = dp4a_ss(a.y, q.y, s); s = dp4a_ss(a.z, q.z, s); s = dp4a_ss(a.w, q.w, s);
    }
    return warp_sum_i(s);
}

// issue the bulk copies of pipeline item `item` into its ring stage (one thread)
__device__ __forceinline__ void issue_item(const Ctx& x, int item, int v0, int v1)
{
    const Params& P = x.P;
    const int st = item % P.stages;
    uint8_t* stage = x.sm + P.s_ring + (size_t)st * P.stage_bytes;
    uint64_t* bar = (uint64_t*)(x.sm + P.s_mbar) + st;
    if (item < P.L) {
        const int* chs = (const int*)(x.sm + P.s_chs);
        const int ch0 = chs[x.c], nch = chs[x.c + 1] - ch0;
        const uint32_t ssm_b = (uint32_t)nch * P.d_state * 4, conv_b = (uint32_t)nch * 16;
        mbar_expect_tx(bar, P.chunk_bytes + ssm_b + conv_b);
        bulk_g2s(stage, P.chunks + ((size_t)item * P.G + x.c) * P.chunk_bytes, P.chunk_bytes, bar);
        if (nch > 0) {
            bulk_g2s(stage + P.st_ssm, P.ssm + (size_t)item * P.ssm_lstride + (size_t)ch0 * P.d_state, ssm_b, bar);
            bulk_g2s(stage + P.st_conv, P.conv + (size_t)item * P.conv_lstride + (size_t)ch0 * 4, conv_b, bar);
        }
    } else {
        const int row0 = v0 + (item - P.L) * P.lm_rows_item;
        const int nrows = min(P.lm_rows_item, v1 - row0);
        const uint32_t bytes = (uint32_t)nrows * P.d_model;
        mbar_expect_tx(bar, bytes);
        bulk_g2s(stage, P.emb + (size_t)row0 * P.d_model, bytes, bar);
    }
}

__device__ __forceinline__ void wait_item(const Ctx& x, int item)
{
    const int st = item % x.P.stages;
    uint64_t* bar = (uint64_t*)(x.sm + x.P.s_mbar) + st;
    const uint32_t parity = (uint32_t)(item / x.P.stages) & 1u;
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > SPIN_LIMIT) { poll_fail(x); break; }
    }
}

// ---- hop (a): publish this CTA's (sum of squares, amax), gather all, derive the quantiser constants ----
__device__ __forceinline__ void exchange_stats(const Ctx& x, uint64_t* buf, uint32_t flag, double ss_own, float amax_own,
                                               int d, float& inv, float& s)
{
    const Params& P = x.P;
    if (x.tid == 0) {
        const long long b = __double_as_longlong(ss_own);
        ll_store(buf + 3 * x.c + 0, ll_pack32((uint32_t)((unsigned long long)b >> 32), flag));
        ll_store(buf + 3 * x.c + 1, ll_pack32((uint32_t)b, flag));
        ll_store(buf + 3 * x.c + 2, ll_pack32(__float_as_uint(amax_own), flag));
    }
    uint32_t* st = (uint32_t*)(x.sm + P.s_stats);
    poll_words<32>(x, buf, 3 * P.G, flag, [&](int idx, uint64_t v) { st[idx] = (uint32_t)v; });
    __syncthreads();
    float* bc = (float*)(x.sm + P.s_red) + 3 * NWARPS;   // behind block_sum_max's scratch
    if (x.wid == 0) {
        double ss = 0.0;
        float am = 0.0f;
        for (int g = x.lane; g < P.G; g += 32) {
            ss += __hiloint2double((int)st[3 * g], (int)st[3 * g + 1]);
            am = fmaxf(am, __uint_as_float(st[3 * g + 2]));
        }
        ss = warp_sum(ss);
        am = warp_max(am);
        if (x.lane == 0) {
            float i_, s_;
            quant_consts(ss, am, d, P.eps, i_, s_);
            bc[0] = i_; bc[1] = s_;
        }
    }
    __syncthreads();
    inv = bc[0];
    s = bc[1];
}

// ---- hop (b): quantise the own slice, publish the codes, gather everyone's codes into xq; returns sum q ----
__device__ __forceinline__ int exchange_codes(const Ctx& x, uint64_t* buf, uint32_t flag8, const float* tq_own, int n_own,
                                              float inv, const int* starts, int wpc, int K, bool canonical)
{
    const Params& P = x.P;
    uint8_t* xq = x.sm + P.s_xq;
    if (x.tid < wpc) {
        uint64_t v = (uint64_t)flag8 << 56;
#pragma unroll
        for (int b = 0; b < CODES_PER_WORD; ++b) {
            const int i = CODES_PER_WORD * x.tid + b;
            if (i < n_own) v |= (uint64_t)(uint8_t)(int8_t)quant_code(tq_own[i], inv) << (8 * b);   // inv == 0 -> code 0
        }
        ll_store(buf + (size_t)x.c * wpc + x.tid, v);
    }
    int qs = 0;
    poll_words<8>(x, buf, P.G * wpc, flag8, [&](int idx, uint64_t v) {
        const int g = idx / wpc, j = idx - g * wpc;
        const int k0 = starts[g], n = starts[g + 1] - k0;
#pragma unroll
        for (int b = 0; b < CODES_PER_WORD; ++b) {
            const int i = CODES_PER_WORD * j + b;
            if (i < n) {
                const int q = (int)(int8_t)(uint8_t)(v >> (8 * b));
                const int k = k0 + i;
                xq[canonical ? k : plane_pos(k, K)] = (uint8_t)q;
                qs += q;
            }
        }
    });
    int* qsum = (int*)((float*)(x.sm + P.s_red) + 3 * NWARPS + 4);
    if (x.tid == 0) *qsum = 0;
    __syncthreads();
    qs = warp_sum_i(qs);
    if (x.lane == 0 && qs != 0) atomicAdd(qsum, qs);
    __syncthreads();
    return *qsum;
}

__global__ void __launch_bounds__(THREADS, 1) k_mega(const Params P)
{
    extern __shared__ __align__(128) uint8_t sm[];
    __shared__ int s_dead;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, c = blockIdx.x;
    Ctx x{ P, sm, tid, lane, wid, c, &s_dead };

    int* chs = (int*)(sm + P.s_chs);
    int* ors = (int*)(sm + P.s_ors);
    uint64_t* mbar = (uint64_t*)(sm + P.s_mbar);
    uint8_t* xq = sm + P.s_xq;
    float* s_bc = (float*)(sm + P.s_bc);
    float* s_u = (float*)(sm + P.s_u);
    float* s_z = (float*)(sm + P.s_z);
    float* s_x = (float*)(sm + P.s_x);
    float* s_tq = (float*)(sm + P.s_tq);
    float* s_vin = (float*)(sm + P.s_vin);
    float* s_vout = (float*)(sm + P.s_vout);
    int* s_acc_in = (int*)(sm + P.s_acc_in);
    int* s_acc_out = (int*)(sm + P.s_acc_out);

    for (int g = tid; g <= P.G; g += THREADS) {
        chs[g] = (int)(((long long)g * P.d_inner) / P.G);
        ors[g] = (int)(((long long)g * P.d_model) / P.G);
    }
    if (tid == 0) {
        s_dead = 0;
        for (int s = 0; s < P.stages; ++s) mbar_init(mbar + s, 1);
        fence_mbar_init();
    }
    __syncthreads();
    const int ch0 = chs[c], nch = chs[c + 1] - ch0;
    const int or0 = ors[c], nor = ors[c + 1] - or0;
    const int v0 = (int)(((long long)c * P.vocab) / P.G), v1 = (int)(((long long)(c + 1) * P.vocab) / P.G);
    const int n_lm_items = (v1 - v0 + P.lm_rows_item - 1) / P.lm_rows_item;
    const int n_items = P.L + n_lm_items;
    if (tid == 0)
        for (int it = 0; it < P.stages && it < n_items; ++it) issue_item(x, it, v0, v1);

    const int ps = P.pos[0] & 3;                     // conv ring slot this step writes
    const int nb = c < P.n_bcdt ? (P.n_bcdt - c + P.G - 1) / P.G : 0;      // early (B|C|dt) rows of this CTA
    const bool taps_on = P.taps != nullptr;

    // LoRA-down rows of this CTA (t = A.xq): row j of t_in belongs to CTA (n_bcdt + j) % G, row j of t_out to
    // CTA (n_bcdt + r + j) % G.  The last warp fetches its row into registers one phase before it is needed.
    const int jt_in = (c - P.n_bcdt % P.G + P.G) % P.G;
    const int jt0 = (c - (P.n_bcdt + P.r) % P.G + 2 * P.G) % P.G;
    int4 pre_in[T_PRE];
    if (wid == NWARPS - 1 && jt_in < P.r && P.L > 0) trow_prefetch(P.A_in + (size_t)jt_in * P.d_model, P.d_model, lane, pre_in);

    // ---------------- S0 embedding + the first norm/quantise, redundantly in every CTA ----------------
    float s_act;                                     // scale of the current activation codes
    int qsum;
    {
        int tok = P.tokens[0];
        if (tok < 0 || tok >= P.vocab) {
            if (tid == 0 && c == 0) atomicOr(P.err, 1);
            tok = tok < 0 ? 0 : P.vocab - 1;
        }
        const int8_t* erow = P.emb + (size_t)tok * P.d_model;
        const float es = P.emb_s[tok];
        double ss = 0.0;
        float amax = 0.0f;
        for (int k = tid; k < P.d_model; k += THREADS) {
            const float u = fmul(es, (float)erow[k]);
            ss = dacc(ss, u, u);
            amax = fmaxf(amax, fabsf(fmul(u, P.first_norm_w[k])));
            if (k >= or0 && k < or0 + nor) s_u[k - or0] = u;
        }
        block_sum_max(x, ss, amax);
        float inv;
        quant_consts(ss, amax, P.d_model, P.eps, inv, s_act);
        int qs = 0;
        const bool canon = P.L == 0;
        for (int k = tid; k < P.d_model; k += THREADS) {
            const float u = fmul(es, (float)erow[k]);
            const int q = amax == 0.0f ? 0 : quant_code(fmul(u, P.first_norm_w[k]), inv);
            xq[canon ? k : plane_pos(k, P.d_model)] = (uint8_t)q;
            qs += q;
        }
        int* qsp = (int*)((float*)(sm + P.s_red) + 3 * NWARPS + 4);
        if (tid == 0) *qsp = 0;
        __syncthreads();
        qs = warp_sum_i(qs);
        if (lane == 0 && qs != 0) atomicAdd(qsp, qs);
        __syncthreads();
        qsum = *qsp;
    }

    // =============================================== layers ===============================================
    for (int l = 0; l < P.L; ++l) {
        const uint32_t f32 = P.base32 + 8u * (uint32_t)l;                   // 32-bit flags of this layer: f32 + hop
        const uint32_t f8 = (uint32_t)((P.e255 * (uint32_t)(P.L + 1) + (uint32_t)l + 1u) % 255u) + 1u;   // codes(u) after layer l
        const uint32_t f8g = (uint32_t)((P.e255 * (uint32_t)(P.L + 1) + (uint32_t)l) % 255u) + 1u;       // codes(g) of layer l
        uint8_t* stage = sm + P.s_ring + (size_t)(l % P.stages) * P.stage_bytes;
        uint8_t* tp = taps_on ? P.taps + (size_t)l * P.tap_lstride : nullptr;
        float* conv_l = P.conv + (size_t)l * P.conv_lstride;
        DFSSM_STAMP(l, 0);
        if (P.prof && tid == 0) P.prof[((size_t)c * (P.L + 1) + l) * PROF_NPH + 15] = globaltimer_ns();

        if (tp && c == 0) {
            for (int k = tid; k < P.d_model; k += THREADS) ((int8_t*)(tp + P.tl.off[0]))[k] = (int8_t)xq[plane_pos(k, P.d_model)];
            if (tid == 0) *(float*)(tp + P.tl.off[1]) = s_act;
        }

        // ---- t_in rows owned by this CTA (warp NWARPS-1): LoRA down-projection on the int8 codes ----
        if (wid == NWARPS - 1) {
            for (int j = jt_in; j < P.r; j += P.G) {
                const int8_t* arow = P.A_in + ((size_t)l * P.r + j) * P.d_model;
                if (j != jt_in) trow_prefetch(arow, P.d_model, lane, pre_in);
                const int t = trow_dot(arow, P.d_model, xq, lane, pre_in);
                if (lane == 0) {
                    ll_store(P.x_t + j, ll_pack32((uint32_t)t, f32 + 0));
                    if (tp) ((int32_t*)(tp + P.tl.off[3]))[j] = t;
                }
            }
        }
        DFSSM_STAMP(l, 1);
        wait_item(x, l);
        DFSSM_STAMP(l, 2);

        // ---- S2: sign rows of this CTA (early rows first, then z, then x), 4 rows per warp pass ----
        {
            const uint32_t* bits = (const uint32_t*)(stage + P.c_in_bits);
            const int n_tasks = nb + 2 * nch;
            for (int q0 = 4 * wid; q0 < n_tasks; q0 += 4 * NWARPS) {
                const uint32_t* rowp[4];
                int slot[4];
                const int nrows = min(4, n_tasks - q0);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int t = q0 + r;
                    slot[r] = t < nb ? 2 * P.nch_max + t : (t < nb + nch ? t - nb : P.nch_max + (t - nb - nch));
                    if (r >= nrows) slot[r] = 0;
                    rowp[r] = bits + (size_t)slot[r] * P.Win;
                }
                const int acc = sign_dot4(rowp, nrows, P.Win, xq, P.d_model, qsum, lane);
                const int r = lane >> 3;
                if ((lane & 7) == 0 && r < nrows) s_acc_in[slot[r]] = acc;
            }
        }
        DFSSM_STAMP(l, 3);
        // ---- gather t_in, v_j = a_s[j] * float(t_j) ----
        {
            const float* a_s = (const float*)(stage + P.c_as_in);
            poll_words<32>(x, P.x_t, P.r, f32 + 0, [&](int j, uint64_t v) { s_vin[j] = fmul(a_s[j], (float)(int32_t)(uint32_t)v); });
        }
        __syncthreads();

        DFSSM_STAMP(l, 4);
        // ---- S3 stage 2 + S4 conv + dt softplus: 4 lanes per row ----
        {
            const int n_rows = 2 * nch + nb;
            const int8_t* Bm = (const int8_t*)(stage + P.c_in_B);
            const float* scale = (const float*)(stage + P.c_in_scale);
            const float* bsv = (const float*)(stage + P.c_in_bs);
            float* ring = (float*)(stage + P.st_conv);
            for (int ib = 0; ib < n_rows; ib += THREADS / 4) {       // warp-uniform trip count (shuffles inside)
                const int i = ib + (tid >> 2), sub = tid & 3;
                const bool valid = i < n_rows;
                int slot = 0, kind = 0, e = 0;     // kind 0 z, 1 x, 2 early
                if (i < nch) { kind = 0; slot = i; }
                else if (i < 2 * nch) { kind = 1; slot = P.nch_max + (i - nch); }
                else if (valid) { kind = 2; slot = 2 * P.nch_max + (i - 2 * nch); e = c + (i - 2 * nch) * P.G; }
                double lo = 0.0;
                const int8_t* brow = Bm + (size_t)slot * P.r_pad;
                if (valid)
                    for (int j = sub; j < P.r; j += 4) lo = dacc(lo, (float)brow[j], s_vin[j]);
                lo += __shfl_xor_sync(0xffffffffu, lo, 1);
                lo += __shfl_xor_sync(0xffffffffu, lo, 2);
                if (sub != 0 || !valid) continue;
                const int acc = s_acc_in[slot];
                const float val = fmul(s_act, fadd(fmul(scale[slot], (float)acc), fmul(bsv[slot], (float)lo)));
                int row;                   // canonical in_proj row (for the taps)
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
                    row = P.d_inner + ch0 + ic;
                    if (tp) ((float*)(tp + P.tl.off[5]))[ch0 + ic] = cv;
                } else {
                    const int ie = i - 2 * nch;
                    row = 2 * P.d_inner + e;
                    float outv;
                    if (e < 2 * P.gs) {        // B or C channel: conv state lives in global memory (4-slot ring)
                        float* rg = conv_l + 4 * (size_t)(P.d_inner + e);
                        const float4 rv = *(const float4*)rg;
                        const float sl[4] = { rv.x, rv.y, rv.z, rv.w };
                        const float s0 = sl[(ps + 1) & 3], s1 = sl[(ps + 2) & 3], s2 = sl[(ps + 3) & 3];
                        const float4 cw = *(const float4*)(stage + P.c_e_conv_w + 16 * ie);
                        float o = ((const float*)(stage + P.c_e_conv_b))[ie];
                        o = ffma(cw.x, s0, o); o = ffma(cw.y, s1, o); o = ffma(cw.z, s2, o); o = ffma(cw.w, val, o);
                        rg[ps] = val;
                        outv = siluf(o);
                        if (tp) ((float*)(tp + P.tl.off[5]))[P.d_inner + e] = outv;
                    } else {                   // dt
                        outv = sp_softplusf(fadd(val, ((const float*)(stage + P.c_e_dtb))[ie]));
                        if (tp) ((float*)(tp + P.tl.off[6]))[e - 2 * P.gs] = outv;
                    }
                    ll_store(P.x_bc + e, ll_pack32(__float_as_uint(outv), f32 + 1));
                }
                if (tp) {
                    ((float*)(tp + P.tl.off[4]))[row] = val;
                    ((int32_t*)(tp + P.tl.off[2]))[row] = acc;
                }
            }
        }
        DFSSM_STAMP(l, 5);
        // ---- gather B' | C' | dt ----
        poll_words<32>(x, P.x_bc, P.n_bcdt, f32 + 1, [&](int e, uint64_t v) { s_bc[e] = __uint_as_float((uint32_t)v); });
        __syncthreads();

        DFSSM_STAMP(l, 6);
        // ---- S5 state update + readout, S6 gate: 16 lanes per channel ----
        double ss_own = 0.0;
        float amax_own = 0.0f;
        {
            const int hpg = P.nheads / P.ngroups;
            const float* alog = (const float*)(stage + P.c_alog);
            const float* Dv = (const float*)(stage + P.c_D);
            const float* gw = (const float*)(stage + P.c_gnorm);
            const int l16 = tid & 15;
            for (int ib = 0; ib < nch; ib += THREADS / 16) {         // warp-uniform trip count (shuffles inside)
                const int i = min(ib + (tid >> 4), nch - 1);
                const bool valid = ib + (tid >> 4) < nch;
                const int ch = ch0 + i, h = ch / P.headdim, grp = h / hpg;
                const float dtv = s_bc[2 * P.gs + h];
                const float An = -sp_expf(alog[i]);
                const float dA = sp_expf(fmul(dtv, An));
                const float xv = s_x[i];
                const float dtx = fmul(dtv, xv);
                float* Hr = (float*)(stage + P.st_ssm) + (size_t)i * P.d_state;
                const float* Bc = s_bc + grp * P.d_state;
                const float* Cc = s_bc + P.gs + grp * P.d_state;
                double a = 0.0;
                for (int n4 = l16; valid && n4 < P.d_state / 4; n4 += 16) {
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
                for (int o = 8; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o, 16);
                if (l16 == 0 && valid) {
                    a = dacc(a, Dv[i], xv);
                    const float y = (float)a;
                    const float gv = fmul(y, siluf(s_z[i]));
                    const float tq = fmul(gv, gw[i]);
                    s_tq[i] = tq;
                    ss_own = dacc(ss_own, gv, gv);
                    amax_own = fmaxf(amax_own, fabsf(tq));
                    if (tp) { ((float*)(tp + P.tl.off[7]))[ch] = y; ((float*)(tp + P.tl.off[8]))[ch] = gv; }
                }
            }
            fence_proxy_async();               // the updated state is about to be read by the async proxy
            block_sum_max(x, ss_own, amax_own);
        }
        DFSSM_STAMP(l, 7);
        // ---- write the state slice back (async), while the exchanges go on ----
        if (tid == 0 && nch > 0) {
            bulk_s2g(P.ssm + (size_t)l * P.ssm_lstride + (size_t)ch0 * P.d_state, stage + P.st_ssm, (uint32_t)nch * P.d_state * 4);
            bulk_s2g(conv_l + (size_t)ch0 * 4, stage + P.st_conv, (uint32_t)nch * 16);
            bulk_commit();
        }
        // t_out row of this CTA: start fetching the LoRA-down row now, use it after the codes arrive
        int4 pre_out[T_PRE];
        if (wid == NWARPS - 1 && jt0 < P.r) trow_prefetch(P.A_out + ((size_t)l * P.r + jt0) * P.d_inner, P.d_inner, lane, pre_out);

        // ---- S6 norm + quantise of g: stats hop, codes hop ----
        float inv_g, s_g;
        exchange_stats(x, P.x_stat3, f32 + 2, ss_own, amax_own, P.d_inner, inv_g, s_g);
        DFSSM_STAMP(l, 8);
        const int qsum_g = exchange_codes(x, P.x_code3, f8g, s_tq, nch, inv_g, chs, P.wpc3, P.d_inner, false);
        if (tp && c == 0) {
            for (int k = tid; k < P.d_inner; k += THREADS) ((int8_t*)(tp + P.tl.off[9]))[k] = (int8_t)xq[plane_pos(k, P.d_inner)];
            if (tid == 0) *(float*)(tp + P.tl.off[10]) = s_g;
        }

        DFSSM_STAMP(l, 9);
        // ---- S7: t_out rows (last warp) and the out_proj sign rows of this CTA ----
        if (wid == NWARPS - 1) {
            for (int j = jt0; j < P.r; j += P.G) {
                const int8_t* arow = P.A_out + ((size_t)l * P.r + j) * P.d_inner;
                if (j != jt0) trow_prefetch(arow, P.d_inner, lane, pre_out);
                const int t = trow_dot(arow, P.d_inner, xq, lane, pre_out);
                if (lane == 0) {
                    ll_store(P.x_t4 + j, ll_pack32((uint32_t)t, f32 + 3));
                    if (tp) ((int32_t*)(tp + P.tl.off[12]))[j] = t;
                }
            }
        }
        {
            const uint32_t* bits = (const uint32_t*)(stage + P.c_out_bits);
            // the last warp is busy with t_out when it owns one: the other warps take the quads first
            for (int q = (wid + 1) % NWARPS; 4 * q < nor; q += NWARPS) {
                const uint32_t* rowp[4];
                const int nrows = min(4, nor - 4 * q);
#pragma unroll
                for (int r = 0; r < 4; ++r) rowp[r] = bits + (size_t)(r < nrows ? 4 * q + r : 0) * P.Wout;
                const int acc = sign_dot4(rowp, nrows, P.Wout, xq, P.d_inner, qsum_g, lane);
                const int r = lane >> 3;
                if ((lane & 7) == 0 && r < nrows) s_acc_out[4 * q + r] = acc;
            }
        }
        DFSSM_STAMP(l, 10);
        {
            const float* a_s = (const float*)(stage + P.c_as_out);
            poll_words<32>(x, P.x_t4, P.r, f32 + 3, [&](int j, uint64_t v) { s_vout[j] = fmul(a_s[j], (float)(int32_t)(uint32_t)v); });
        }
        __syncthreads();

        DFSSM_STAMP(l, 11);
        // ---- S7 epilogue + residual; stats of the new u for the next norm ----
        double ss_u = 0.0;
        float amax_u = 0.0f;
        {
            const int8_t* Bm = (const int8_t*)(stage + P.c_out_B);
            const float* scale = (const float*)(stage + P.c_out_scale);
            const float* bsv = (const float*)(stage + P.c_out_bs);
            const float* nw = (const float*)(stage + P.c_nnorm);
            for (int ib = 0; ib < nor; ib += THREADS / 4) {
                const int i = ib + (tid >> 2), sub = tid & 3;
                const bool valid = i < nor;
                double lo = 0.0;
                const int8_t* brow = Bm + (size_t)(valid ? i : 0) * P.r_pad;
                if (valid)
                    for (int j = sub; j < P.r; j += 4) lo = dacc(lo, (float)brow[j], s_vout[j]);
                lo += __shfl_xor_sync(0xffffffffu, lo, 1);
                lo += __shfl_xor_sync(0xffffffffu, lo, 2);
                if (sub != 0 || !valid) continue;
                const int acc = s_acc_out[i];
                const float o = fmul(s_g, fadd(fmul(scale[i], (float)acc), fmul(bsv[i], (float)lo)));
                const float un = fadd(s_u[i], o);
                s_u[i] = un;
                const float tq = fmul(un, nw[i]);
                s_tq[i] = tq;
                ss_u = dacc(ss_u, un, un);
                amax_u = fmaxf(amax_u, fabsf(tq));
                if (tp) { ((float*)(tp + P.tl.off[13]))[or0 + i] = un; ((int32_t*)(tp + P.tl.off[11]))[or0 + i] = acc; }
            }
            block_sum_max(x, ss_u, amax_u);     // also: every thread is done with this stage's weights
        }
        DFSSM_STAMP(l, 12);
        // ---- refill this ring stage with the item `stages` ahead ----
        if (tid == 0) {
            bulk_wait_read0();                  // the state write-back has finished reading the stage
            if (l + P.stages < n_items) issue_item(x, l + P.stages, v0, v1);
        }
        if (wid == NWARPS - 1 && jt_in < P.r && l + 1 < P.L)
            trow_prefetch(P.A_in + ((size_t)(l + 1) * P.r + jt_in) * P.d_model, P.d_model, lane, pre_in);
        // ---- S1 of the next layer (or S8's norm): stats hop, codes hop ----
        float inv_u;
        exchange_stats(x, P.x_stat1, f32 + 4, ss_u, amax_u, P.d_model, inv_u, s_act);
        DFSSM_STAMP(l, 13);
        qsum = exchange_codes(x, P.x_code1, f8, s_tq, nor, inv_u, ors, P.wpc1, P.d_model, l == P.L - 1);
        DFSSM_STAMP(l, 14);
    }

    // =============================================== S8 LM head ===============================================
    for (int i = tid; i < nor; i += THREADS) P.u_out[or0 + i] = s_u[i];
    DFSSM_STAMP(P.L, 0);
    if (P.prof && tid == 0) P.prof[((size_t)c * (P.L + 1) + P.L) * PROF_NPH + 15] = globaltimer_ns();
    float best = -INFINITY;
    int besti = 0x7fffffff;
    for (int it = 0; it < n_lm_items; ++it) {
        const int item = P.L + it;
        wait_item(x, item);
        const uint8_t* stage = sm + P.s_ring + (size_t)(item % P.stages) * P.stage_bytes;
        const int row0 = v0 + it * P.lm_rows_item;
        const int nrows_it = min(P.lm_rows_item, v1 - row0);
        const int nchunk = P.d_model >> 4;
        for (int q0 = 4 * wid; q0 < nrows_it; q0 += 4 * NWARPS) {
            const int nr = min(4, nrows_it - q0);
            int s[4] = { 0, 0, 0, 0 };
            for (int ch = lane; ch < nchunk; ch += 32) {
                const int4 q4 = *(const int4*)(xq + 16 * ch);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    if (r < nr) {
                        const int4 a4 = *(const int4*)(stage + (size_t)(q0 + r) * P.d_model + 16 * ch);
                        s[r] = dp4a_ss(a4.x, q4.x, s[r]); s[r] = dp4a_ss(a4.y, q4.y, s[r]);
                        s[r] = dp4a_ss(a4.z, q4.z, s[r]); s[r] = dp4a_ss(a4.w, q4.w, s[r]);
                    }
                }
            }
            const bool up16 = (lane & 16) != 0, up8 = (lane & 8) != 0;
            int k0 = up16 ? s[2] : s[0], k1 = up16 ? s[3] : s[1];
            const int t0 = up16 ? s[0] : s[2], t1 = up16 ? s[1] : s[3];
            k0 += __shfl_xor_sync(0xffffffffu, t0, 16);
            k1 += __shfl_xor_sync(0xffffffffu, t1, 16);
            int v = up8 ? k1 : k0;
            const int sv = up8 ? k0 : k1;
            v += __shfl_xor_sync(0xffffffffu, sv, 8);
            v += __shfl_xor_sync(0xffffffffu, v, 4);
            v += __shfl_xor_sync(0xffffffffu, v, 2);
            v += __shfl_xor_sync(0xffffffffu, v, 1);
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
        float* rv = (float*)(sm + P.s_red);
        int* ri = (int*)(rv + NWARPS);
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
            s_last = prev == (unsigned)P.G - 1;
            bulk_wait0();                       // all state write-backs of this CTA are complete
        }
        __syncthreads();
        if (s_last && wid == 0) {
            __threadfence();
            float b = -INFINITY;
            int bi = 0x7fffffff;
            for (int g = lane; g < P.G; g += 32) {
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
