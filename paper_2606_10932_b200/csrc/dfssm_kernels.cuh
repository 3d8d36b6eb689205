// Kernel-chain implementation of the DF-SSM decode step ("chain" path): one kernel per row of
// the step list in include/dfssm.h, replayed as one CUDA graph.  Works for any batch.
// The fused persistent kernel for small batches lives in dfssm_mega.cuh.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "dfssm_math.cuh"

namespace dfssm {

// Programmatic dependent launch (launch_pdl in dfssm_api.cu): wait until the kernel in front of this one in the chain has completed
// and its writes are visible, then let the kernel behind this one be scheduled.  Everything a kernel reads from or writes to
// buffers of the chain comes after this call; loads of weights (and of the SSM state, which only the same layer's kernel of the
// step before wrote) may come before it.  A no-op for a launch without the attribute.
__device__ __forceinline__ void pdl_wait()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");      // behind the wait: at most two kernels of the chain overlap
}


// ---- device-side view of one layer's weights (pointers into the arena copy of the blob) ----
struct LayerW {
    const float* norm_w;
    const uint32_t* in_sign; const __half* in_row_scale;
    const int8_t* in_A; const float* in_a_s; const int8_t* in_B; const float* in_b_s;
    const float* conv_w; const float* conv_b;
    const float* A_log; const float* dt_bias; const float* D;
    const float* gnorm_w;
    const uint32_t* out_sign; const __half* out_row_scale;
    const int8_t* out_A; const float* out_a_s; const int8_t* out_B; const float* out_b_s;
};

struct Dims {
    int n_layers, d_model, d_inner, headdim, d_state, ngroups, vocab, r;
    int nheads, d_in_proj, conv_dim;
    float eps;
    int fmt;          // weight format variants (R25): bit 0 = 17-level scaffold (five bit planes), bit 1 = int4 LoRA
};

// debug taps: byte offsets inside one (layer, seq) record; stride = off[DFSSM_TAP_COUNT]
struct TapLayout { uint32_t off[16]; };

constexpr int T_STRIDE = 64;      // ints per sequence in the LoRA stage-1 buffer t
constexpr int PROJ_BT = 8;        // sequences per CTA tile in the projection kernels
constexpr int SSM_PB = 16;        // (head, p) rows per CTA in the SSM kernel

// =============================================================================================
// S0  embedding: u = e_s[tok] * float(E[tok,:])
// =============================================================================================
__global__ void k_embed(const int32_t* __restrict__ tokens, const int8_t* __restrict__ E,
                        const float* __restrict__ e_s, int vocab, int d, float* __restrict__ u,
                        int* __restrict__ err)
{
    const int b = blockIdx.y;
    int tok = tokens[b];
    if (tok < 0 || tok >= vocab) {
        if (threadIdx.x == 0 && blockIdx.x == 0) atomicOr(err, 1);
        tok = tok < 0 ? 0 : vocab - 1;
    }
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < d) u[(size_t)b * d + k] = fmul(e_s[tok], (float)E[(size_t)tok * d + k]);
}

// =============================================================================================
// S1 / S6(b) / S8(a)  RMSNorm + per-token absmax int8 quantiser (R4, R13)
//   rstd = 1/sqrt(mean(v^2)+eps); t_k = v_k*w_k; amax = max|t_k|; q_k = clamp(rint(t_k*(127/amax)));
//   s = (amax*rstd)/127.  Writes the codes twice: canonical order (xq) and the bit-plane order
//   (xqp) the masked-dp4a sign dot product reads: inside each group of 32, canonical position
//   8j+i goes to position 4i+j.  Also writes sum_k q_k (the sign dot needs 2*P - sum q).
//   One CTA per sequence.
// =============================================================================================
constexpr int NQ_THREADS = 512;

__global__ void __launch_bounds__(NQ_THREADS)
k_normquant(const float* __restrict__ v, int ldv, const float* __restrict__ w, int d, float eps,
            int8_t* __restrict__ xq, int8_t* __restrict__ xqp, int ldq, float* __restrict__ s_out,
            int32_t* __restrict__ qsum_out, uint8_t* __restrict__ taps, uint32_t tap_stride,
            uint32_t tap_q_off, uint32_t tap_s_off,
            int32_t* __restrict__ zero_acc = nullptr, int ld_acc = 0, int32_t* __restrict__ zero_t = nullptr)
{
    // up to NQ_R elements per thread stay in registers between the two passes; their norm weights are read before pdl_wait
    constexpr int NQ_R = 8;
    const bool in_regs = d <= NQ_R * NQ_THREADS;
    float wv[NQ_R], tv[NQ_R];
    if (in_regs) {
#pragma unroll
        for (int i = 0; i < NQ_R; ++i) {
            const int k = threadIdx.x + i * NQ_THREADS;
            wv[i] = k < d ? w[k] : 0.0f;
        }
    }
    pdl_wait();
    // the split-K tensor-core projection that follows adds into acc / t: this sequence's rows are zeroed here (their last
    // reader ran before this kernel) instead of by two memset nodes per projection
    if (zero_acc) {
        int32_t* za = zero_acc + (size_t)blockIdx.x * ld_acc;
        for (int k = threadIdx.x; k < ld_acc; k += NQ_THREADS) za[k] = 0;
        if (threadIdx.x < T_STRIDE) zero_t[(size_t)blockIdx.x * T_STRIDE + threadIdx.x] = 0;
    }
    __shared__ double sh_d[NQ_THREADS / 32];
    __shared__ float sh_f[NQ_THREADS / 32];
    __shared__ int sh_i[NQ_THREADS / 32];
    __shared__ float sh_bcast[2];
    const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const float* vb = v + (size_t)b * ldv;

    double ss = 0.0;
    float amax = 0.0f;
    if (in_regs) {
#pragma unroll
        for (int i = 0; i < NQ_R; ++i) {
            const int k = tid + i * NQ_THREADS;
            const float x = k < d ? vb[k] : 0.0f;          // (a zero adds +0 to the sum and 0 to the maximum)
            ss = dacc(ss, x, x);
            tv[i] = fmul(x, wv[i]);
            amax = fmaxf(amax, fabsf(tv[i]));
        }
    } else {
        for (int k = tid; k < d; k += NQ_THREADS) {
            const float x = vb[k];
            ss = dacc(ss, x, x);
            amax = fmaxf(amax, fabsf(fmul(x, w[k])));
        }
    }
    ss = warp_sum(ss);
    amax = warp_max(amax);
    if (lane == 0) { sh_d[wid] = ss; sh_f[wid] = amax; }
    __syncthreads();
    if (wid == 0) {
        double s2 = lane < NQ_THREADS / 32 ? sh_d[lane] : 0.0;
        float m2 = lane < NQ_THREADS / 32 ? sh_f[lane] : 0.0f;
        s2 = warp_sum(s2);
        m2 = warp_max(m2);
        if (lane == 0) {
            const float ms = (float)(s2 / (double)d);
            const float rstd = fdiv(1.0f, __fsqrt_rn(fadd(ms, eps)));
            sh_bcast[0] = m2;
            sh_bcast[1] = rstd;
        }
    }
    __syncthreads();
    amax = sh_bcast[0];
    const float rstd = sh_bcast[1];
    const float inv = amax == 0.0f ? 0.0f : fdiv(127.0f, amax);
    const float s = amax == 0.0f ? 0.0f : fdiv(fmul(amax, rstd), 127.0f);
    int qs = 0;
    int8_t* qb = xq + (size_t)b * ldq;
    int8_t* qpb = xqp + (size_t)b * ldq;
    uint8_t* tp = taps ? taps + (size_t)b * tap_stride : nullptr;
    auto emit = [&](int k, float tk) {
        const int q = amax == 0.0f ? 0 : quant_code(tk, inv);
        qs += q;
        qb[k] = (int8_t)q;
        if (xqp) {                                         // plane order and code sum: only the dp4a sign rows read them
            const int p = k & 31;
            qpb[(k & ~31) + 4 * (p & 7) + (p >> 3)] = (int8_t)q;
        }
        if (tp) ((int8_t*)(tp + tap_q_off))[k] = (int8_t)q;
    };
    if (in_regs) {
#pragma unroll
        for (int i = 0; i < NQ_R; ++i) {
            const int k = tid + i * NQ_THREADS;
            if (k < d) emit(k, tv[i]);
        }
    } else {
        for (int k = tid; k < d; k += NQ_THREADS) emit(k, fmul(vb[k], w[k]));
    }
    if (!qsum_out) {                                       // tensor-core projections behind this kernel: no code sum needed
        if (tid == 0) {
            s_out[b] = s;
            if (tp) *(float*)(tp + tap_s_off) = s;
        }
        return;
    }
    qs = warp_sum_i(qs);
    if (lane == 0) sh_i[wid] = qs;
    __syncthreads();
    if (tid == 0) {
        int tot = 0;
        for (int i = 0; i < NQ_THREADS / 32; ++i) tot += sh_i[i];
        qsum_out[b] = tot;
        s_out[b] = s;
        if (tp) *(float*)(tp + tap_s_off) = s;
    }
}

// =============================================================================================
// S2 + S3 stage 1 (and S7): bit-packed sign matvec + int8 LoRA down-projection, exact int32.
//   rows [0, rows)      : acc_i = sum_k sign_ik * q_k = 2 * sum_{bit_ik = 1} q_k - sum_k q_k
//   rows [rows, rows+r) : t_j   = sum_k A_jk * q_k
//   One warp per row; a lane takes whole 32-bit sign words.  For each word the eight masks
//   0x01010101 << i pick bit i of every byte; dp4a(u8 mask bytes, s8 codes) against the codes
//   stored in bit-plane order gives 2^i * (partial sum); the eight partial sums are recombined
//   exactly as sum_i a_i * 2^(7-i) = 128 * P.
//   grid = (row blocks, batch tiles of PROJ_BT); dynamic smem = PROJ_BT * 2 * K bytes.
// =============================================================================================
constexpr int PROJ_THREADS = 256;

__global__ void __launch_bounds__(PROJ_THREADS)
k_proj(const uint32_t* __restrict__ sign, const int8_t* __restrict__ A, int rows, int r, int K,
       const int8_t* __restrict__ xq, const int8_t* __restrict__ xqp, int ldq,
       const int32_t* __restrict__ qsum, int batch, int32_t* __restrict__ acc, int ld_acc,
       int32_t* __restrict__ t)
{
    pdl_wait();
    extern __shared__ __align__(16) uint8_t smem[];
    const int b0 = blockIdx.y * PROJ_BT;
    const int nb = min(PROJ_BT, batch - b0);
    int8_t* sq = (int8_t*)smem;                    // [nb][K] canonical
    int8_t* sqp = sq + (size_t)PROJ_BT * K;        // [nb][K] bit-plane order
    for (int i = threadIdx.x; i < nb * (K / 16); i += PROJ_THREADS) {
        const int bb = i / (K / 16), c = i % (K / 16);
        ((int4*)sq)[bb * (K / 16) + c] = ((const int4*)(xq + (size_t)(b0 + bb) * ldq))[c];
        ((int4*)sqp)[bb * (K / 16) + c] = ((const int4*)(xqp + (size_t)(b0 + bb) * ldq))[c];
    }
    __syncthreads();

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int W = K / 32;
    const int rows_total = rows + r;
    for (int row = blockIdx.x * (PROJ_THREADS / 32) + wid; row < rows_total;
         row += gridDim.x * (PROJ_THREADS / 32)) {
        if (row < rows) {
            const uint32_t* wrow = sign + (size_t)row * W;
            int p128[PROJ_BT];
#pragma unroll
            for (int bb = 0; bb < PROJ_BT; ++bb) p128[bb] = 0;
            for (int w = lane; w < W; w += 32) {
                const uint32_t bits = __ldg(wrow + w);
#pragma unroll
                for (int bb = 0; bb < PROJ_BT; ++bb) {
                    if (bb < nb) {
                        const int4 qa = *(const int4*)(sqp + (size_t)bb * K + 32 * w);
                        const int4 qb = *(const int4*)(sqp + (size_t)bb * K + 32 * w + 16);
                        int a;
                        a = dp4a_us(bits & 0x01010101u, qa.x, 0) * 128;
                        a += dp4a_us(bits & 0x02020202u, qa.y, 0) * 64;
                        a += dp4a_us(bits & 0x04040404u, qa.z, 0) * 32;
                        a += dp4a_us(bits & 0x08080808u, qa.w, 0) * 16;
                        a += dp4a_us(bits & 0x10101010u, qb.x, 0) * 8;
                        a += dp4a_us(bits & 0x20202020u, qb.y, 0) * 4;
                        a += dp4a_us(bits & 0x40404040u, qb.z, 0) * 2;
                        a += dp4a_us(bits & 0x80808080u, qb.w, 0);
                        p128[bb] += a;
                    }
                }
            }
#pragma unroll
            for (int bb = 0; bb < PROJ_BT; ++bb) {
                if (bb < nb) {
                    const int p = warp_sum_i(p128[bb]) / 128;    // exact: every term is a multiple of 128
                    if (lane == 0) acc[(size_t)(b0 + bb) * ld_acc + row] = 2 * p - qsum[b0 + bb];
                }
            }
        } else {
            const int j = row - rows;
            const int4* arow = (const int4*)(A + (size_t)j * K);
            int s[PROJ_BT];
#pragma unroll
            for (int bb = 0; bb < PROJ_BT; ++bb) s[bb] = 0;
            for (int c = lane; c < K / 16; c += 32) {
                const int4 a4 = __ldg(arow + c);
#pragma unroll
                for (int bb = 0; bb < PROJ_BT; ++bb) {
                    if (bb < nb) {
                        const int4 q4 = *(const int4*)(sq + (size_t)bb * K + 16 * c);
                        int a = s[bb];
                        a = dp4a_ss(a4.x, q4.x, a);
                        a = dp4a_ss(a4.y, q4.y, a);
                        a = dp4a_ss(a4.z, q4.z, a);
                        a = dp4a_ss(a4.w, q4.w, a);
                        s[bb] = a;
                    }
                }
            }
#pragma unroll
            for (int bb = 0; bb < PROJ_BT; ++bb) {
                if (bb < nb) {
                    const int tot = warp_sum_i(s[bb]);
                    if (lane == 0) t[(size_t)(b0 + bb) * T_STRIDE + j] = tot;
                }
            }
        }
    }
}

// S3 stage 2 + dequantisation for one output row (Eq. 3; R6, R7):
//   out = s_x * ( w_s[i]*float(acc_i) + b_s[i]*float( sum_j float(B_ij) * v_j ) ),  v_j = a_s[j]*float(t_j)
// the sum over j runs in binary64, in index order, and is rounded once.
__device__ __forceinline__ float proj_epilogue_row(int acc_i, const __half* __restrict__ row_scale,
                                                   const int8_t* __restrict__ B,
                                                   const float* __restrict__ b_s, int i, int r,
                                                   const float* v_sh, float s_x)
{
    double lo = 0.0;
    const int8_t* brow = B + (size_t)i * r;
    for (int j = 0; j < r; ++j) lo = dacc(lo, (float)brow[j], v_sh[j]);
    const float lo_f = (float)lo;
    const float m1 = fmul(__half2float(row_scale[i]), (float)acc_i);
    const float m2 = fmul(b_s[i], lo_f);
    return fmul(s_x, fadd(m1, m2));
}

constexpr int SSM_THREADS = 256;

// four consecutive state values: fp32 state, or the fp16 state format of DESIGN.md R24 (stored as binary16, RN-even of the
// binary32 update; the readout of the step uses the unrounded binary32 values)
__device__ __forceinline__ float4 state_ld4(const float* p) { return *(const float4*)p; }
__device__ __forceinline__ void state_st4(float* p, float4 v) { *(float4*)p = v; }
__device__ __forceinline__ float4 state_ld4(const __half* p)
{
    const uint2 r = *(const uint2*)p;
    const __half2 a = *(const __half2*)&r.x, b = *(const __half2*)&r.y;
    return make_float4(__low2float(a), __high2float(a), __low2float(b), __high2float(b));
}
__device__ __forceinline__ void state_st4(__half* p, float4 v)
{
    const __half2 a = __halves2half2(__float2half_rn(v.x), __float2half_rn(v.y)), b = __halves2half2(__float2half_rn(v.z), __float2half_rn(v.w));
    uint2 r;
    r.x = *(const uint32_t*)&a;
    r.y = *(const uint32_t*)&b;
    *(uint2*)p = r;
}

// =============================================================================================
// S3 stage 2 + S4 conv + SiLU / softplus for EVERY in_proj row, once per sequence (the streaming state kernel below reads
// finished values only):  fin[b] = [ silu(z) : d_inner ][ silu(conv(x | B | C)) : conv_dim ][ dt : nheads ][ dA : nheads ]
//   grid = (ceil(d_in_proj / FIN_THREADS), batch).  Same arithmetic, value by value, as the persistent kernel's in_proj epilogue.
// =============================================================================================
constexpr int FIN_THREADS = 128;

__global__ void __launch_bounds__(FIN_THREADS)
k_fin(LayerW L, Dims dm, const int32_t* __restrict__ acc, int ld_acc, const int32_t* __restrict__ t,
      const float* __restrict__ s_x, float* __restrict__ conv_ring, const int32_t* __restrict__ pos,
      float* __restrict__ fin, uint8_t* __restrict__ taps, uint32_t tap_stride, TapLayout tl)
{
    pdl_wait();
    __shared__ float v_sh[64];
    const int b = blockIdx.y, tid = threadIdx.x;
    const int gs = dm.ngroups * dm.d_state, d_in_proj = 2 * dm.d_inner + 2 * gs + dm.nheads;
    if (tid < dm.r) v_sh[tid] = fmul(L.in_a_s[tid], (float)t[(size_t)b * T_STRIDE + tid]);
    __syncthreads();
    const int row = blockIdx.x * FIN_THREADS + tid;
    if (row >= d_in_proj) return;
    uint8_t* tp = taps ? taps + (size_t)b * tap_stride : nullptr;
    float* out = fin + (size_t)b * (d_in_proj + dm.nheads);
    const float val = proj_epilogue_row(acc[(size_t)b * ld_acc + row], L.in_row_scale, L.in_B, L.in_b_s, row, dm.r, v_sh, s_x[b]);
    if (tp) ((float*)(tp + tl.off[4]))[row] = val;                               // ZXBCDT
    if (row < dm.d_inner) {
        out[row] = siluf(val);                                                   // the gate factor of S6
    } else if (row < d_in_proj - dm.nheads) {
        const int ps = pos[b] & 3;
        const int c = row - dm.d_inner;                                          // conv channel
        float* ring = conv_ring + ((size_t)b * dm.conv_dim + c) * 4;
        const float4 rg = *(const float4*)ring;
        const float sl[4] = { rg.x, rg.y, rg.z, rg.w };
        const float s0 = sl[(ps + 1) & 3], s1 = sl[(ps + 2) & 3], s2 = sl[(ps + 3) & 3];
        const float4 cw = *(const float4*)(L.conv_w + 4 * (size_t)c);
        float o = L.conv_b[c];
        o = ffma(cw.x, s0, o);
        o = ffma(cw.y, s1, o);
        o = ffma(cw.z, s2, o);
        o = ffma(cw.w, val, o);
        ring[ps] = val;
        const float cv = siluf(o);
        if (tp) ((float*)(tp + tl.off[5]))[c] = cv;                              // XBC_CONV
        out[row] = cv;
    } else {
        const int h = row - (d_in_proj - dm.nheads);
        const float dtv = sp_softplusf(fadd(val, L.dt_bias[h]));
        if (tp) ((float*)(tp + tl.off[6]))[h] = dtv;                             // DT
        out[row] = dtv;
        out[row + dm.nheads] = sp_expf(fmul(dtv, -sp_expf(L.A_log[h])));         // dA (Eq. 5)
    }
}

// k_fin for lora_rank = 4 * JW (JW = 2, 4, 8, 16): four lanes share a row's LoRA sum, each holding its JW values of v in
// registers and reading its JW bytes of the row with one load (a warp reads 8 x 32 contiguous bytes per pass); a CTA of
// FIN_THREADS threads finishes FIN_THREADS rows in 4 passes, then lane `sub` of a group finishes the row of pass `sub`, so that
// the row epilogues (conv, SiLU, softplus) run on every lane and row = base + tid is coalesced.  fp64 sum, tree (p0+p1)+(p2+p3).
template <int JW> struct BytesT;
template <> struct BytesT<1> { using T = uint8_t; };
template <> struct BytesT<2> { using T = uint16_t; };
template <> struct BytesT<4> { using T = uint32_t; };
template <> struct BytesT<8> { using T = uint2; };
template <> struct BytesT<16> { using T = uint4; };

// LoRA stage 2 of FIN_THREADS consecutive rows (from `base`) by one CTA, lora_rank = 4 * JW: returns, in every thread, the
// binary64 sum  sum_j float(B[row][j]) * v_j,  v_j = a_s[j] * float(t_j),  of row = base + threadIdx.x (0 beyond n_rows).
// Lane `sub` of a group of four holds v_j for its JW values of j and reads its JW bytes of a row with one load; the group
// walks through its four rows, and the tree of the sum is (p0 + p1) + (p2 + p3).  No shared memory, no barrier.
// I4: the matrix holds int4 pairs (format variant, R25): a lane's JW values are JW / 2 bytes, element 2i = low nibble.
// Two halves, so that the weight half can run before pdl_wait(): lora_load4 reads the lane's bytes of its group's four rows and
// its JW scales a_s; lora_sum4 makes v from the (dependent) t and sums.
template <int JW, bool I4> struct LoraRegs {
    typename BytesT<I4 ? JW / 2 : JW>::T w[4];
    float as[JW];
};
template <int JW, bool I4>
__device__ __forceinline__ void lora_load4(const int8_t* __restrict__ B, const float* __restrict__ a_s, int base, int n_rows, LoraRegs<JW, I4>& R)
{
    constexpr int RK = 4 * JW;
    const int q = threadIdx.x >> 2, sub = threadIdx.x & 3;
    using WT = typename BytesT<I4 ? JW / 2 : JW>::T;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int rk = min(base + q * 4 + k, n_rows - 1);          // rows beyond the end are summed and never used
        R.w[k] = *(const WT*)((const uint8_t*)B + ((size_t)rk * RK + sub * JW) / (I4 ? 2 : 1));
    }
#pragma unroll
    for (int i = 0; i < JW; ++i) R.as[i] = a_s[sub * JW + i];
}
template <int JW, bool I4>
__device__ __forceinline__ double lora_sum4(const LoraRegs<JW, I4>& R, const int32_t* __restrict__ t_row)
{
    const int sub = threadIdx.x & 3;
    double v[JW];
#pragma unroll
    for (int i = 0; i < JW; ++i) v[i] = (double)fmul(R.as[i], (float)t_row[sub * JW + i]);
    double part[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        double lo = 0.0;
        const uint8_t* wb = (const uint8_t*)&R.w[k];
#pragma unroll
        for (int i = 0; i < JW; ++i) {
            if constexpr (I4) {
                const int nib = (wb[i >> 1] >> (4 * (i & 1))) & 0xf;
                lo = __fma_rn((double)((nib ^ 8) - 8), v[i], lo);
            } else {
                lo = __fma_rn((double)(int)(int8_t)wb[i], v[i], lo);
            }
        }
        lo += __shfl_xor_sync(0xffffffffu, lo, 1);
        lo += __shfl_xor_sync(0xffffffffu, lo, 2);
        part[k] = lo;
    }
    return sub == 0 ? part[0] : sub == 1 ? part[1] : sub == 2 ? part[2] : part[3];
}
template <int JW, bool I4 = false>
__device__ __forceinline__ double lora_up4(const int8_t* __restrict__ B, const float* __restrict__ a_s,
                                           const int32_t* __restrict__ t_row, int base, int n_rows)
{
    LoraRegs<JW, I4> R;
    lora_load4<JW, I4>(B, a_s, base, n_rows, R);
    return lora_sum4<JW, I4>(R, t_row);
}

template <int JW, bool I4 = false>
__global__ void __launch_bounds__(FIN_THREADS)
k_fin4(LayerW L, Dims dm, const int32_t* __restrict__ acc, int ld_acc, const int32_t* __restrict__ t,
       const float* __restrict__ s_x, float* __restrict__ conv_ring, const int32_t* __restrict__ pos,
       float* __restrict__ fin, uint8_t* __restrict__ taps, uint32_t tap_stride, TapLayout tl)
{
    const int b = blockIdx.y, tid = threadIdx.x;
    const int gs = dm.ngroups * dm.d_state, d_in_proj = 2 * dm.d_inner + 2 * gs + dm.nheads;
    const int base = blockIdx.x * FIN_THREADS;
    const int row = base + tid;                                  // the row this lane finishes
    const bool own = row < d_in_proj;

    // requested early: everything the row epilogue needs - the weights before pdl_wait (they do not depend on the kernel in front)
    const int rl = own ? row : 0;
    const float rs = __half2float(L.in_row_scale[rl]), bs = L.in_b_s[rl];
    const bool is_conv = own && row >= dm.d_inner && row < d_in_proj - dm.nheads;
    const int c = is_conv ? row - dm.d_inner : 0;                // conv channel
    float* ring = conv_ring + ((size_t)b * dm.conv_dim + c) * 4;
    float4 rg = make_float4(0.f, 0.f, 0.f, 0.f), cw = rg;
    float cb = 0.f;
    if (is_conv) {
        cw = *(const float4*)(L.conv_w + 4 * (size_t)c);
        cb = L.conv_b[c];
    }
    LoraRegs<JW, I4> lr;
    lora_load4<JW, I4>(L.in_B, L.in_a_s, base, d_in_proj, lr);
    // also before the wait: what kernels further back than the one in front wrote (at most two kernels of the chain overlap, so
    // those have completed): the scale of k_normquant, the conv ring and the ring position of the step before
    const float sx = s_x[b];
    if (is_conv) rg = *(const float4*)ring;
    const int ps = pos[b] & 3;
    pdl_wait();
    const int acc_i = acc[(size_t)b * ld_acc + rl];

    const double lo = lora_sum4<JW, I4>(lr, t + (size_t)b * T_STRIDE);
    if (!own) return;
    uint8_t* tp = taps ? taps + (size_t)b * tap_stride : nullptr;
    float* out = fin + (size_t)b * (d_in_proj + dm.nheads);
    const float val = fmul(sx, fadd(fmul(rs, (float)acc_i), fmul(bs, (float)lo)));
    if (tp) ((float*)(tp + tl.off[4]))[row] = val;                               // ZXBCDT
    if (row < dm.d_inner) {
        out[row] = siluf(val);                                                   // the gate factor of S6
    } else if (is_conv) {
        const float sl[4] = { rg.x, rg.y, rg.z, rg.w };
        const float s0 = sl[(ps + 1) & 3], s1 = sl[(ps + 2) & 3], s2 = sl[(ps + 3) & 3];
        float o = cb;
        o = ffma(cw.x, s0, o);
        o = ffma(cw.y, s1, o);
        o = ffma(cw.z, s2, o);
        o = ffma(cw.w, val, o);
        ring[ps] = val;
        const float cv = siluf(o);
        if (tp) ((float*)(tp + tl.off[5]))[c] = cv;                              // XBC_CONV
        out[row] = cv;
    } else {
        const int h = row - (d_in_proj - dm.nheads);
        const float dtv = sp_softplusf(fadd(val, L.dt_bias[h]));
        if (tp) ((float*)(tp + tl.off[6]))[h] = dtv;                             // DT
        out[row] = dtv;
        out[row + dm.nheads] = sp_expf(fmul(dtv, -sp_expf(L.A_log[h])));         // dA (Eq. 5)
    }
}

// =============================================================================================
// S5 state update + readout + S6 gate on finished inputs (k_fin): a pure stream over the state.
//   grid = (headdim / PB, nheads, batch); every load of the CTA is issued before its only barrier.
//   DS = d_state at compile time (no bounds checks, no tail loop: the kernel is issue-bound once the prologue is gone), 0 = any.
// =============================================================================================
#ifndef DFSSM_SSM_MINB
#define DFSSM_SSM_MINB 5
#endif
template <int PB, int DS, typename ST>
__global__ void __launch_bounds__(SSM_THREADS, DFSSM_SSM_MINB)
k_ssm_stream(LayerW L, Dims dm, const float* __restrict__ fin, ST* __restrict__ ssm /* [batch][h][p][n] */,
             float* __restrict__ g /* [batch][d_inner] */, uint8_t* __restrict__ taps, uint32_t tap_stride, TapLayout tl)
{
    extern __shared__ __align__(16) uint8_t smem[];
    const int ds = DS ? DS : dm.d_state;
    float* Bc = (float*)smem;                      // [d_state]
    float* Cc = Bc + ds;                           // [d_state]
    constexpr int LANES = SSM_THREADS / PB;        // lanes per state row
    const int b = blockIdx.z, h = blockIdx.y, p0 = blockIdx.x * PB;
    const int grp = dm.ngroups == 1 ? 0 : h / (dm.nheads / dm.ngroups);
    const int tid = threadIdx.x;
    const int gs = dm.ngroups * ds, d_in_proj = 2 * dm.d_inner + 2 * gs + dm.nheads;
    const float* src = fin + (size_t)b * (d_in_proj + dm.nheads);

    const int p = tid / LANES, l16 = tid % LANES;
    const int ch = h * dm.headdim + p0 + p;
    ST* Hr = ssm + ((size_t)b * dm.d_inner + ch) * ds;
    constexpr int H_PRE = DS ? DS / 4 / LANES : 32 / LANES;    // chunks held in registers; with DS = 0 further ones are loaded late
    static_assert(!DS || DS % (4 * LANES) == 0, "d_state must be a multiple of 4 * lanes per row");
    float4 hpre[H_PRE];
#pragma unroll
    for (int j = 0; j < H_PRE; ++j) {
        const int n4 = l16 + LANES * j;
        if (DS || n4 < ds / 4) hpre[j] = state_ld4(Hr + 4 * n4);
    }
    const float Dh = L.D[h];
    pdl_wait();                                    // the state was requested above: only this layer's kernel of the step before wrote it
    const float xv = src[dm.d_inner + ch];
    const float dtv = src[d_in_proj - dm.nheads + h], dA = src[d_in_proj + h];
    const float sz = src[ch];                      // silu(z) from k_fin
    for (int i = tid; i < ds; i += SSM_THREADS) {
        Bc[i] = src[2 * dm.d_inner + grp * ds + i];
        Cc[i] = src[2 * dm.d_inner + gs + grp * ds + i];
    }
    __syncthreads();

    const float dtx = fmul(dtv, xv);
    double a = 0.0;
#pragma unroll
    for (int j = 0; j < H_PRE; ++j) {
        const int n4 = l16 + LANES * j;
        if (!DS && n4 >= ds / 4) break;
        float4 hv = hpre[j];
        const float4 bv = *(const float4*)(Bc + 4 * n4);
        const float4 cv = *(const float4*)(Cc + 4 * n4);
        hv.x = ffma(dA, hv.x, fmul(dtx, bv.x));
        hv.y = ffma(dA, hv.y, fmul(dtx, bv.y));
        hv.z = ffma(dA, hv.z, fmul(dtx, bv.z));
        hv.w = ffma(dA, hv.w, fmul(dtx, bv.w));
        state_st4(Hr + 4 * n4, hv);
        a = dacc(a, cv.x, hv.x);
        a = dacc(a, cv.y, hv.y);
        a = dacc(a, cv.z, hv.z);
        a = dacc(a, cv.w, hv.w);
    }
    if (!DS) {
        for (int n4 = l16 + LANES * H_PRE; n4 < ds / 4; n4 += LANES) {
            float4 hv = state_ld4(Hr + 4 * n4);
            const float4 bv = *(const float4*)(Bc + 4 * n4);
            const float4 cv = *(const float4*)(Cc + 4 * n4);
            hv.x = ffma(dA, hv.x, fmul(dtx, bv.x));
            hv.y = ffma(dA, hv.y, fmul(dtx, bv.y));
            hv.z = ffma(dA, hv.z, fmul(dtx, bv.z));
            hv.w = ffma(dA, hv.w, fmul(dtx, bv.w));
            state_st4(Hr + 4 * n4, hv);
            a = dacc(a, cv.x, hv.x);
            a = dacc(a, cv.y, hv.y);
            a = dacc(a, cv.z, hv.z);
            a = dacc(a, cv.w, hv.w);
        }
    }
#pragma unroll
    for (int o = LANES / 2; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o, LANES);
    if (l16 == 0) {
        a = dacc(a, Dh, xv);
        const float y = (float)a;
        const float gv = fmul(y, sz);
        g[(size_t)b * dm.d_inner + ch] = gv;
        if (taps) {
            uint8_t* tp = taps + (size_t)b * tap_stride;
            ((float*)(tp + tl.off[7]))[ch] = y;
            ((float*)(tp + tl.off[8]))[ch] = gv;
        }
    }
}

// =============================================================================================
// S7 epilogue + residual: u_i <- u_i + s_g*( w_s[i]*acc_i + b_s[i]*lo_i )
// =============================================================================================
constexpr int EPI_THREADS = 128;

__global__ void __launch_bounds__(EPI_THREADS)
k_epi_out(LayerW L, int d_model, int r, const int32_t* __restrict__ acc, int ld_acc,
          const int32_t* __restrict__ t, const float* __restrict__ s_g, float* __restrict__ u,
          uint8_t* __restrict__ taps, uint32_t tap_stride, uint32_t tap_hidden_off)
{
    pdl_wait();
    __shared__ float v_sh[64];
    const int b = blockIdx.y;
    if (threadIdx.x < r) v_sh[threadIdx.x] = fmul(L.out_a_s[threadIdx.x], (float)t[(size_t)b * T_STRIDE + threadIdx.x]);
    __syncthreads();
    const int i = blockIdx.x * EPI_THREADS + threadIdx.x;
    if (i >= d_model) return;
    const float o = proj_epilogue_row(acc[(size_t)b * ld_acc + i], L.out_row_scale, L.out_B, L.out_b_s, i, r,
                                      v_sh, s_g[b]);
    const float un = fadd(u[(size_t)b * d_model + i], o);
    u[(size_t)b * d_model + i] = un;
    if (taps) ((float*)(taps + (size_t)b * tap_stride + tap_hidden_off))[i] = un;
}

// k_epi_out for lora_rank = 4 * JW: the LoRA sum by lora_up4 (four lanes per row, vector loads of the LoRA-up bytes)
template <int JW, bool I4 = false>
__global__ void __launch_bounds__(FIN_THREADS)
k_epi_out4(LayerW L, int d_model, const int32_t* __restrict__ acc, int ld_acc,
           const int32_t* __restrict__ t, const float* __restrict__ s_g, float* __restrict__ u,
           uint8_t* __restrict__ taps, uint32_t tap_stride, uint32_t tap_hidden_off)
{
    const int b = blockIdx.y, base = blockIdx.x * FIN_THREADS, i = base + threadIdx.x;
    const bool own = i < d_model;
    const int il = own ? i : 0;
    const float rs = __half2float(L.out_row_scale[il]), bs = L.out_b_s[il];      // weights: before pdl_wait
    LoraRegs<JW, I4> lr;
    lora_load4<JW, I4>(L.out_B, L.out_a_s, base, d_model, lr);
    const float sg = s_g[b];                               // k_normquant(g): two kernels back, complete (see k_fin4)
    const float u0 = u[(size_t)b * d_model + il];          // the layer before
    pdl_wait();
    const int acc_i = acc[(size_t)b * ld_acc + il];
    const double lo = lora_sum4<JW, I4>(lr, t + (size_t)b * T_STRIDE);
    if (!own) return;
    const float o = fmul(sg, fadd(fmul(rs, (float)acc_i), fmul(bs, (float)lo)));
    const float un = fadd(u0, o);
    u[(size_t)b * d_model + i] = un;
    if (taps) ((float*)(taps + (size_t)b * tap_stride + tap_hidden_off))[i] = un;
}

// k_epi_out4 fused with the RMSNorm + quantiser that follows it (S7 of layer l, then S1 of layer l + 1 or S8(a)): the CTAs of one
// sequence form a thread-block cluster (d_model / blockDim.x <= 8 CTAs), exchange their partial sum of squares and maximum through
// distributed shared memory and quantise their own elements, so the separate k_normquant launch (one CTA per sequence, 5 us) goes.
// Tensor-core chain without taps only; d_model % blockDim.x == 0.  w_next: norm weights of the sub-layer that follows.
// zero_acc / zero_t as in k_normquant (this sequence's rows, zeroed once every CTA of the cluster has read them).
constexpr int EPN_MAX_THREADS = 512;
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

template <int JW, bool I4 = false>
__global__ void __launch_bounds__(EPN_MAX_THREADS)
k_epi_norm4(LayerW L, int d_model, const int32_t* acc, int ld_acc, const int32_t* t,
            const float* s_g, float* __restrict__ u, const float* __restrict__ w_next, float eps,
            int8_t* __restrict__ xq, int ldq, float* s_out, int32_t* zero_acc, int32_t* zero_t)      // s_out may be s_g, zero_acc / zero_t are acc / t
{
    __shared__ double sh_d[EPN_MAX_THREADS / 32];
    __shared__ float sh_f[EPN_MAX_THREADS / 32];
    __shared__ double cl_ss;                 // this CTA's partials, read by every CTA of the cluster
    __shared__ float cl_amax;
    __shared__ float sh_bcast[2];
    const int b = blockIdx.y, nthr = blockDim.x, base = blockIdx.x * nthr, tid = threadIdx.x, i = base + tid;
    const int lane = tid & 31, wid = tid >> 5, ncta = gridDim.x, rank = blockIdx.x;
    const float rs = __half2float(L.out_row_scale[i]), bs = L.out_b_s[i];      // weights: before pdl_wait
    const float wn = w_next[i];
    LoraRegs<JW, I4> lr;
    lora_load4<JW, I4>(L.out_B, L.out_a_s, base, d_model, lr);
    const float sg = s_g[b];                               // k_normquant(g): two kernels back, complete (see k_fin4)
    const float u0 = u[(size_t)b * d_model + i];           // the layer before
    pdl_wait();
    const int acc_i = acc[(size_t)b * ld_acc + i];
    const double lo = lora_sum4<JW, I4>(lr, t + (size_t)b * T_STRIDE);
    const float o = fmul(sg, fadd(fmul(rs, (float)acc_i), fmul(bs, (float)lo)));
    const float un = fadd(u0, o);
    u[(size_t)b * d_model + i] = un;
    // ---- the norm of what follows: partials of this CTA ----
    const float tk = fmul(un, wn);
    double ss = warp_sum(dacc(0.0, un, un));
    float amax = warp_max(fabsf(tk));
    if (lane == 0) { sh_d[wid] = ss; sh_f[wid] = amax; }
    __syncthreads();
    if (wid == 0) {
        double s2 = lane < nthr / 32 ? sh_d[lane] : 0.0;
        float m2 = lane < nthr / 32 ? sh_f[lane] : 0.0f;
        s2 = warp_sum(s2);
        m2 = warp_max(m2);
        if (lane == 0) { cl_ss = s2; cl_amax = m2; }
    }
    cluster_arrive();
    cluster_wait();                          // every CTA of the sequence has published its partials and read its acc / t
    if (wid == 0) {
        double s2 = 0.0;
        float m2 = 0.0f;
        if (lane < ncta) {
            uint32_t ra, rb;
            asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"((uint32_t)__cvta_generic_to_shared(&cl_ss)), "r"(lane));
            asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rb) : "r"((uint32_t)__cvta_generic_to_shared(&cl_amax)), "r"(lane));
            asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(s2) : "r"(ra) : "memory");
            asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(m2) : "r"(rb) : "memory");
        }
        s2 = warp_sum(s2);
        m2 = warp_max(m2);
        if (lane == 0) {
            const float ms = (float)(s2 / (double)d_model);
            sh_bcast[0] = m2;
            sh_bcast[1] = fdiv(1.0f, __fsqrt_rn(fadd(ms, eps)));
        }
    }
    __syncthreads();
    cluster_arrive();                        // this CTA has read its peers; it leaves only when they have read it (wait at the end)
    amax = sh_bcast[0];
    const float rstd = sh_bcast[1];
    const float inv = amax == 0.0f ? 0.0f : fdiv(127.0f, amax);
    xq[(size_t)b * ldq + i] = (int8_t)(amax == 0.0f ? 0 : quant_code(tk, inv));
    if (rank == 0 && tid == 0) s_out[b] = amax == 0.0f ? 0.0f : fdiv(fmul(amax, rstd), 127.0f);
    if (zero_acc) {                          // rows of the split-K projection that follows
        int32_t* za = zero_acc + (size_t)b * ld_acc;
        const int per = (ld_acc + ncta - 1) / ncta, k1 = min(ld_acc, (rank + 1) * per);
        for (int k = rank * per + tid; k < k1; k += nthr) za[k] = 0;
        if (rank == 0 && tid < T_STRIDE) zero_t[(size_t)b * T_STRIDE + tid] = 0;
    }
    cluster_wait();
}

// debug-only: copy int32 vectors into the taps (acc, t)
__global__ void k_tap_copy_i32(const int32_t* __restrict__ src, int ld_src, int n, uint8_t* __restrict__ taps,
                               uint32_t tap_stride, uint32_t off)
{
    const int b = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) ((int32_t*)(taps + (size_t)b * tap_stride + off))[i] = src[(size_t)b * ld_src + i];
}

// =============================================================================================
// S8  tied int8 LM head on the quantised final hidden (R16):
//   logit_v = float( sum_k E_vk * hq_k ) * (s_h * e_s[v]);  one warp per vocabulary row.
// =============================================================================================
constexpr int LM_THREADS = 256;

__global__ void __launch_bounds__(LM_THREADS)
k_lmhead(const int8_t* __restrict__ E, const float* __restrict__ e_s, int vocab, int K,
         const int8_t* __restrict__ xq, int ldq, const float* __restrict__ s_h, int batch,
         float* __restrict__ logits)
{
    pdl_wait();
    extern __shared__ __align__(16) uint8_t smem[];
    const int b0 = blockIdx.y * PROJ_BT;
    const int nb = min(PROJ_BT, batch - b0);
    int8_t* sq = (int8_t*)smem;
    for (int i = threadIdx.x; i < nb * (K / 16); i += LM_THREADS) {
        const int bb = i / (K / 16), c = i % (K / 16);
        ((int4*)sq)[bb * (K / 16) + c] = ((const int4*)(xq + (size_t)(b0 + bb) * ldq))[c];
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int row = blockIdx.x * (LM_THREADS / 32) + wid; row < vocab; row += gridDim.x * (LM_THREADS / 32)) {
        const int4* erow = (const int4*)(E + (size_t)row * K);
        int s[PROJ_BT];
#pragma unroll
        for (int bb = 0; bb < PROJ_BT; ++bb) s[bb] = 0;
        for (int c = lane; c < K / 16; c += 32) {
            const int4 a4 = __ldg(erow + c);
#pragma unroll
            for (int bb = 0; bb < PROJ_BT; ++bb) {
                if (bb < nb) {
                    const int4 q4 = *(const int4*)(sq + (size_t)bb * K + 16 * c);
                    int a = s[bb];
                    a = dp4a_ss(a4.x, q4.x, a);
                    a = dp4a_ss(a4.y, q4.y, a);
                    a = dp4a_ss(a4.z, q4.z, a);
                    a = dp4a_ss(a4.w, q4.w, a);
                    s[bb] = a;
                }
            }
        }
        const float es = e_s[row];
#pragma unroll
        for (int bb = 0; bb < PROJ_BT; ++bb) {
            if (bb < nb) {
                const int tot = warp_sum_i(s[bb]);
                if (lane == 0) logits[(size_t)(b0 + bb) * vocab + row] = fmul((float)tot, fmul(s_h[b0 + bb], es));
            }
        }
    }
}

// greedy token: argmax with the lowest index on ties; also advances the conv ring position
constexpr int AM_THREADS = 1024;

__global__ void __launch_bounds__(AM_THREADS)
k_argmax(const float* __restrict__ logits, int vocab, int32_t* __restrict__ next, int32_t* __restrict__ tok,
         int32_t* __restrict__ pos, int pos_inc = 1)
{
    pdl_wait();
    __shared__ float sv[AM_THREADS / 32];
    __shared__ int si[AM_THREADS / 32];
    const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const float* lg = logits + (size_t)b * vocab;
    float best = -INFINITY;
    int bi = 0x7fffffff;
    for (int i = tid; i < vocab; i += AM_THREADS) {
        const float x = lg[i];
        if (x > best || (x == best && i < bi)) { best = x; bi = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, best, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
    }
    if (lane == 0) { sv[wid] = best; si[wid] = bi; }
    __syncthreads();
    if (wid == 0) {
        best = sv[lane];
        bi = si[lane];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
        }
        if (lane == 0) {
            next[b] = bi == 0x7fffffff ? 0 : bi;
            tok[b] = next[b];                      // the next step's input if the caller decodes greedily
            pos[b] = (pos[b] + pos_inc) & 3;
        }
    }
}

// =============================================================================================
// Temperature / top-k sampling of the next token (R23; the generation loop of P:126), one CTA per sequence:
//   ranks 0 .. k-1 = the k largest logits, equal logits by lower index first (k rounds of a CTA-wide argmax over the
//   candidates that come strictly after the previous pick in that order); w_r = sp_expf((l_r - l_0) / temperature);
//   c_r = fp64 running sum in rank order; the pick is the smallest r with c_r > u * c_{k-1}.  u[b] in [0,1) comes from the caller.
//   Overwrites next[b] and tok[b] (the next dfssm_step's input); the conv ring position is NOT touched (the step did that).
// =============================================================================================
constexpr int SAMPLE_THREADS = 1024, SAMPLE_KMAX = 64;

__global__ void __launch_bounds__(SAMPLE_THREADS)
k_sample(const float* __restrict__ logits, int vocab, float temperature, int top_k, const float* __restrict__ u,
         int32_t* __restrict__ next, int32_t* __restrict__ tok)
{
    __shared__ float sv[SAMPLE_THREADS / 32];
    __shared__ int si[SAMPLE_THREADS / 32];
    __shared__ float pick_v[SAMPLE_KMAX];
    __shared__ int pick_i[SAMPLE_KMAX];
    const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const float* lg = logits + (size_t)b * vocab;
    if (top_k < 1) top_k = 1;
    if (top_k > vocab) top_k = vocab;
    if (top_k > SAMPLE_KMAX) top_k = SAMPLE_KMAX;
    if (!(temperature > 0.0f)) top_k = 1;
    float prev_v = 0.0f;
    int prev_i = -1;
    for (int r = 0; r < top_k; ++r) {
        float best = 0.0f;
        int bi = 0x7fffffff;
        for (int i = tid; i < vocab; i += SAMPLE_THREADS) {
            const float x = lg[i];
            if (r > 0 && !(x < prev_v || (x == prev_v && i > prev_i))) continue;
            if (bi == 0x7fffffff || x > best) { best = x; bi = i; }      // ascending i per thread: the lowest index wins among equals
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (oi != 0x7fffffff && (bi == 0x7fffffff || ov > best || (ov == best && oi < bi))) { best = ov; bi = oi; }
        }
        if (lane == 0) { sv[wid] = best; si[wid] = bi; }
        __syncthreads();
        if (wid == 0) {
            best = sv[lane];
            bi = si[lane];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const float ov = __shfl_xor_sync(0xffffffffu, best, o);
                const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (oi != 0x7fffffff && (bi == 0x7fffffff || ov > best || (ov == best && oi < bi))) { best = ov; bi = oi; }
            }
            if (lane == 0) { pick_v[r] = best; pick_i[r] = bi; }
        }
        __syncthreads();
        prev_v = pick_v[r];
        prev_i = pick_i[r];
    }
    if (tid == 0) {
        int choice = pick_i[0];
        if (top_k > 1) {
            double c[SAMPLE_KMAX];
            double run = 0.0;
            for (int r = 0; r < top_k; ++r) {
                const float w = sp_expf(fdiv(fadd(pick_v[r], -pick_v[0]), temperature));
                run += (double)w;
                c[r] = run;
            }
            const double thr = (double)u[b] * run;
            choice = pick_i[top_k - 1];
            for (int r = 0; r < top_k; ++r)
                if (c[r] > thr) { choice = pick_i[r]; break; }
        }
        next[b] = choice;
        tok[b] = choice;
    }
}

}  // namespace dfssm
