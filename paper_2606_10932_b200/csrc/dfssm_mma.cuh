// Batched projections (batch >= 16) on the 5th-generation tensor cores: S2 + S3 stage 1 (and S7) as
//   [rows + r] x K   times   K x batch      int8 x int8 -> int32      (BJ north_star; S.8(a) last row)
// The +-1 scaffold tile is unpacked from its sign bits into int8 in shared memory (never in HBM), the LoRA-down rows are
// appended as further int8 rows of the same tile, the activation codes are the N operand, and the int32 accumulators
// live in TMEM: tcgen05.mma.kind::i8, M = 128, N = 64, K = 32 per instruction, issued by one thread; tcgen05.commit ->
// mbarrier tells the CTA that the shared-memory tile may be overwritten; tcgen05.ld brings the accumulators back.
// The tied int8 LM head (S8) is the same contraction with the embedding rows as the int8 rows and a float epilogue.
// Integer arithmetic: exact, so the results are bit-identical to the dp4a path (k_proj).
//
// Shared-memory operand layout (K-major, no swizzle; "core matrix" = 8 rows x 16 bytes, stored contiguously):
//   offset(row m, byte k) = (k / 16) * LBO + (m / 8) * 128 + (m % 8) * 16 + k % 16,   LBO = (tile rows / 8) * 128, SBO = 128
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "dfssm_kernels.cuh"

namespace dfssm {
namespace mma {

constexpr int TM = 128;            // rows of the weight tile (MMA M)
constexpr int TN = 64;             // sequences per tile (MMA N)
constexpr int KC = 256;            // bytes of K per shared-memory stage (8 MMAs of K = 32); K itself may be any multiple of KMULT
constexpr int KMULT = 128;         // (a last half stage is filled with zeros)
constexpr int THREADS = 512;
constexpr uint32_t LBO_A = (TM / 8) * 128, LBO_B = (TN / 8) * 128, SBO = 128;
constexpr uint32_t SPIN_LIMIT = 1u << 22;
constexpr int STAGES = 2;                                  // shared-memory stages: the unpack of chunk k + 1 runs under the MMAs of chunk k
constexpr size_t SMEM_BYTES = (size_t)STAGES * (TM + TN) * KC;    // dynamic shared memory of k_proj_mma

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// shared-memory matrix descriptor (sm_100): start address, leading / stride byte offsets in 16-byte units, version 1, no swizzle
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) | ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) |
           (1ull << 46);
}
// instruction descriptor of kind::i8: D = s32, A = B = signed 8-bit, both K-major, N >> 3 at bit 17, M >> 4 at bit 24
constexpr uint32_t IDESC = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TN >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);

// 4 sign bits -> 4 bytes of +1 (bit 1) / -1 (bit 0)
__device__ __forceinline__ uint32_t signs4(uint32_t bits)
{
    const uint32_t spread = ((bits & 0xfu) * 0x00204081u) & 0x01010101u;
    return 0xffffffffu ^ (spread * 0xfeu);
}

// ---- format variants (R25) ----
// 17-level scaffold: four weights (bits sh .. sh+3 of the five planes of one 32-weight word) -> four int8 levels m - 8 in [-8, 8]
__device__ __forceinline__ uint32_t spread4(uint32_t bits) { return ((bits & 0xfu) * 0x00204081u) & 0x01010101u; }
__device__ __forceinline__ uint32_t levels4(const uint32_t* pl, int sh)
{
    const uint32_t m = spread4(pl[0] >> sh) + (spread4(pl[1] >> sh) << 1) + (spread4(pl[2] >> sh) << 2) + (spread4(pl[3] >> sh) << 3) +
                       (spread4(pl[4] >> sh) << 4);              // bytes 0 .. 16: no carry between bytes
    return __vsub4(m, 0x08080808u);
}
// int4 LoRA: eight two's-complement nibbles (element 2i = low nibble of byte i) -> eight int8 in element order
__device__ __forceinline__ uint2 nibbles8(uint32_t w)
{
    const uint32_t lo = w & 0x0f0f0f0fu, hi = (w >> 4) & 0x0f0f0f0fu;
    const uint32_t a = __byte_perm(lo, hi, 0x5140), b = __byte_perm(lo, hi, 0x7362);
    return make_uint2(__vsub4(a ^ 0x08080808u, 0x08080808u), __vsub4(b ^ 0x08080808u, 0x08080808u));
}

// grid = (ceil((rows + r) / 128), ceil(batch / 64), ksplit); 512 threads; K % 128 == 0.  LM head: rows = 0, r = vocab,
// A = the embedding, ksplit = 1, logits / s_h / e_s given.  With ksplit > 1 every CTA takes a
// slice of K and ADDS its int32 partial sums into acc / t (exact in any order), which the caller has zeroed.
// 16 warps: the kernel was bound by the issue latency of 4 warps that unpack, stage and store in turn (ncu: 11 % of the warp
// slots, one issue per 8 cycles per warp); a thread now unpacks 32 weights and stages 16 codes per chunk, and a warp reads one
// 32-lane x 16-column block of the accumulators.
// FMT: bit 0 = `sign` holds the five bit planes of the 17-level scaffold ([row][K/32][5]), bit 1 = `A` holds int4 pairs ([r][K/2]).
template <int FMT>
__global__ void __launch_bounds__(THREADS)
k_proj_mma(const uint32_t* __restrict__ sign, const int8_t* __restrict__ A, int rows, int r, int K,
           const int8_t* __restrict__ xq, int ldq, int batch, int32_t* __restrict__ acc, int ld_acc,
           int32_t* __restrict__ t, int* __restrict__ err,
           float* __restrict__ logits = nullptr, const float* __restrict__ s_h = nullptr, const float* __restrict__ e_s = nullptr)
{
    extern __shared__ __align__(128) uint8_t stage_mem[];     // [STAGES][ A tile TM x KC | B tile TN x KC ]
    __shared__ __align__(8) uint64_t mbar[STAGES];
    __shared__ uint32_t tmem_base;
    const int tid = threadIdx.x, wid = tid >> 5, lane = tid & 31;
    const int row0 = blockIdx.x * TM, b0 = blockIdx.y * TN;
    const int rows_total = rows + r;
    const int W = K / 32;

    if (wid == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base)), "r"((uint32_t)TN) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&mbar[s])) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = tmem_base;

    // unpack: thread = (K quarter qk, tile row am): 64 weights = the four 16-byte K columns 4 qk .. 4 qk + 3 of row am; a warp
    // writes 32 consecutive rows of one column (512 contiguous bytes of shared memory)
    const int am = tid & (TM - 1), qk = tid >> 7;
    const int urow = row0 + am;                        // the weight row this thread unpacks
    // stage: thread = (16-byte pieces xc and xc + 8, sequence bn)
    const int bn = tid & (TN - 1), xc = tid >> 6;
    const bool b_valid = b0 + bn < batch;
    const uint32_t a_off = (uint32_t)(4 * qk) * LBO_A + (am >> 3) * 128 + (am & 7) * 16;
    const uint32_t b_off = TM * KC + (uint32_t)xc * LBO_B + (bn >> 3) * 128 + (bn & 7) * 16;
    bool dead = false;
    // waits until the MMAs committed to mbar[s] in phase `parity` have read their stage; a thread that timed out stops waiting
    // (it still runs through every barrier of the loop, so the CTA stays in step) and the failure is reported at the end
    auto wait_stage = [&](int s, uint32_t parity) {
        uint32_t spins = 0, ok = 0;
        while (!ok && !dead) {
            asm volatile(
                "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                : "=r"(ok) : "r"(smem_u32(&mbar[s])), "r"(parity) : "memory");
            if (!ok && ++spins > SPIN_LIMIT) dead = true;
        }
    };

    const int nchunk = (K + KC - 1) / KC, kc0 = (int)(((long long)blockIdx.z * nchunk) / gridDim.z), kc1 = (int)(((long long)(blockIdx.z + 1) * nchunk) / gridDim.z);
    const bool split = gridDim.z > 1;
    // the sign words and the codes of a stage are requested one stage ahead (registers), before the stage in hand is unpacked,
    // so that their latency runs under the unpack and the MMAs; the few LoRA-down rows (last tile only) are read directly
    const bool is_sign = urow < rows;
    constexpr int PL = (FMT & 1) ? 5 : 1;               // words per 32 weights
    constexpr int NWD = 2 * PL;                         // words of this thread per stage (64 weights)
    const uint32_t* sign_row = sign + ((size_t)(is_sign ? urow : 0) * W + 2 * qk) * PL;
    const int8_t* x_row = xq + (size_t)(b_valid ? b0 + bn : 0) * ldq + xc * 16;
    uint32_t w_next[NWD], w_cur[NWD];
#pragma unroll
    for (int i = 0; i < NWD; ++i) w_next[i] = 0;
    uint4 x_next[2] = { make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0) }, x_cur[2];
    uint4 a_next[4] = { make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0) }, a_cur[4];
    auto request_w = [&](int kc) {     // the weights: independent of the kernel in front
        const int ka = kc * KC + qk * 64;      // byte offset of this thread's piece inside K; beyond K (last half stage) the operands are zero
#pragma unroll
        for (int i = 0; i < NWD / 2; ++i) {
            const uint2 ww = (is_sign && ka < K) ? *(const uint2*)(sign_row + (size_t)kc * (KC / 32) * PL + 2 * i) : make_uint2(0, 0);
            w_next[2 * i] = ww.x;
            w_next[2 * i + 1] = ww.y;
        }
        if (!is_sign && urow < rows_total && ka < K) {      // int8 / int4 rows (LoRA-down, the LM head's embedding): a stage ahead as well
            if (FMT & 2) {
                const uint4* src = (const uint4*)((const uint8_t*)A + ((size_t)(urow - rows) * K + ka) / 2);
                a_next[0] = src[0]; a_next[1] = src[1];
            } else {
                const uint4* src = (const uint4*)(A + (size_t)(urow - rows) * K + ka);
#pragma unroll
                for (int c = 0; c < 4; ++c) a_next[c] = src[c];
            }
        }
    };
    auto request_x = [&](int kc) {     // the codes: written by the kernel in front
        const int kx = kc * KC + xc * 16;
        x_next[0] = (b_valid && kx < K) ? *(const uint4*)(x_row + kc * KC) : make_uint4(0, 0, 0, 0);
        x_next[1] = (b_valid && kx + 128 < K) ? *(const uint4*)(x_row + kc * KC + 128) : make_uint4(0, 0, 0, 0);
    };
    auto request = [&](int kc) { request_w(kc); request_x(kc); };
    // TMEM allocation, barrier initialisation and the first weight request run under the kernel in front
    const bool early_w = kc0 < kc1;
    if (early_w) request_w(kc0);
    pdl_wait();
    if (kc0 < kc1) {
        if (!early_w) request_w(kc0);
        request_x(kc0);
    }
    for (int kc = kc0; kc < kc1; ++kc) {
        const int it = kc - kc0, s = it % STAGES, use = it / STAGES;
        uint8_t* a_dst = stage_mem + (size_t)s * (TM + TN) * KC + a_off;
        uint8_t* b_dst = stage_mem + (size_t)s * (TM + TN) * KC + b_off;
#pragma unroll
        for (int i = 0; i < NWD; ++i) w_cur[i] = w_next[i];
        x_cur[0] = x_next[0]; x_cur[1] = x_next[1];
#pragma unroll
        for (int c = 0; c < 4; ++c) a_cur[c] = a_next[c];
        if (kc + 1 < kc1) request(kc + 1);
        if (use > 0) wait_stage(s, (uint32_t)(use - 1) & 1u);           // the MMAs that read this stage last are done
        // ---- A: 64 weights of this row -> int8 ----
        const bool a_in = kc * KC + qk * 64 < K;
        if ((FMT & 1) && is_sign && a_in) {              // 17 levels: word j of the stage = planes w_cur[5 j .. 5 j + 4]
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const uint32_t* pl = w_cur + 5 * (c >> 1);
                const int sh = 16 * (c & 1);
                *(uint4*)(a_dst + c * LBO_A) = make_uint4(levels4(pl, sh), levels4(pl, sh + 4), levels4(pl, sh + 8), levels4(pl, sh + 12));
            }
        } else if (is_sign && a_in) {
            const uint32_t w0 = w_cur[0], w1 = w_cur[1 % NWD];
            *(uint4*)a_dst = make_uint4(signs4(w0), signs4(w0 >> 4), signs4(w0 >> 8), signs4(w0 >> 12));
            *(uint4*)(a_dst + LBO_A) = make_uint4(signs4(w0 >> 16), signs4(w0 >> 20), signs4(w0 >> 24), signs4(w0 >> 28));
            *(uint4*)(a_dst + 2 * LBO_A) = make_uint4(signs4(w1), signs4(w1 >> 4), signs4(w1 >> 8), signs4(w1 >> 12));
            *(uint4*)(a_dst + 3 * LBO_A) = make_uint4(signs4(w1 >> 16), signs4(w1 >> 20), signs4(w1 >> 24), signs4(w1 >> 28));
        } else if ((FMT & 2) && !is_sign && urow < rows_total && a_in) {      // int4 LoRA-down row: 64 values in 32 bytes
            const uint4 p0 = a_cur[0], p1 = a_cur[1];
            const uint32_t pw[8] = { p0.x, p0.y, p0.z, p0.w, p1.x, p1.y, p1.z, p1.w };
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const uint2 e0 = nibbles8(pw[2 * c]), e1 = nibbles8(pw[2 * c + 1]);
                *(uint4*)(a_dst + c * LBO_A) = make_uint4(e0.x, e0.y, e1.x, e1.y);
            }
        } else if (!is_sign && urow < rows_total && a_in) {
#pragma unroll
            for (int c = 0; c < 4; ++c) *(uint4*)(a_dst + c * LBO_A) = a_cur[c];
        } else {
#pragma unroll
            for (int c = 0; c < 4; ++c) *(uint4*)(a_dst + c * LBO_A) = make_uint4(0, 0, 0, 0);
        }
        // ---- B: 2 x 16 codes of one sequence ----
        *(uint4*)b_dst = x_cur[0];
        *(uint4*)(b_dst + 8 * LBO_B) = x_cur[1];
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the tensor core
        __syncthreads();
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
            for (int j = 0; j < KC / 32; ++j) {
                const uint32_t sbase = smem_u32(stage_mem) + (uint32_t)s * (TM + TN) * KC;
                const uint64_t da = smem_desc(sbase + j * 2 * LBO_A, LBO_A, SBO);
                const uint64_t db = smem_desc(sbase + TM * KC + j * 2 * LBO_B, LBO_B, SBO);
                const uint32_t accumulate = (kc > kc0 || j > 0) ? 1u : 0u;
                asm volatile(
                    "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                    "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %6, %7, %8}, p;\n\t}"
                    ::"r"(tmem), "l"(da), "l"(db), "r"(IDESC), "r"(accumulate), "r"(0u), "r"(0u), "r"(0u), "r"(0u) : "memory");
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&mbar[s])) : "memory");
        }
    }
    // ---- the last commit covers every MMA before it: wait for it, then read the accumulators ----
    if (kc1 > kc0) {
        const int it = kc1 - 1 - kc0;
        wait_stage(it % STAGES, (uint32_t)(it / STAGES) & 1u);
    }
    if (dead) atomicOr(err, 4);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

    // ---- epilogue: TMEM lane = row of the tile, column = sequence; warp = (lane quarter wid % 4, 16 columns wid / 4) ----
    if (!__syncthreads_or(dead ? 1 : 0) && kc1 > kc0) {
        const int grow = row0 + (wid & 3) * 32 + lane, cg = wid >> 2;
        const bool is_acc = grow < rows, is_t = !is_acc && grow < rows_total;
        uint32_t v[16];
        const uint32_t taddr = tmem + ((uint32_t)((wid & 3) * 32) << 16) + (uint32_t)(cg * 16);
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
            : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
              "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
            : "r"(taddr) : "memory");
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int b = b0 + cg * 16 + i;
            if (b < batch) {
                if (logits) {          // S8: logit_v = float(acc_v) * (s_h * e_s[v])   (R16); rows == 0, r == vocab
                    if (is_t) logits[(size_t)b * r + grow] = fmul((float)(int32_t)v[i], fmul(s_h[b], e_s[grow]));
                    continue;
                }
                int32_t* dst = is_acc ? acc + (size_t)b * ld_acc + grow : t + (size_t)b * T_STRIDE + (grow - rows);
                if (is_acc || is_t) {
                    if (split) atomicAdd(dst, (int32_t)v[i]);
                    else *dst = (int32_t)v[i];
                }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (wid == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"((uint32_t)TN) : "memory");
}

}  // namespace mma
}  // namespace dfssm
