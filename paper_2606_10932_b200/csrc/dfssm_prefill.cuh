// Prefill (P:112, P:416 feed prompts in chunks): T prompt positions of ONE sequence per call, layer by layer.
// The projections run over the T positions as a batch (weights read once per chunk: k_normquant, k_proj / k_proj_mma, k_epi_out of
// the chain path with "batch" = T); what couples the positions -- the 4-tap conv and the state recurrence -- runs in the kernels
// below, serial in t where the method is: the arithmetic is, operation for operation, that of T calls of dfssm_step (same
// proj_epilogue_row, same conv chain, same h <- fma(dA, h, (dt x) B) and fp64 readout), so the result is bit-identical to feeding
// the prompt through the step path (tests/test_gpu_prefill.py).  The chunked SSD scan of the paper (block_len 64) re-associates
// the recurrence and is NOT what is built here (R22).
#pragma once
#include "dfssm_kernels.cuh"

namespace dfssm {
namespace prefill {

constexpr int CHUNK = 128;            // positions per chunk (activation buffers are sized for it)

// S3 stage 2 for ALL in_proj rows of all positions: zx[t][i] = s_x[t] * (w_s[i]*acc[t][i] + b_s[i]*sum_j B_ij v_j[t])
constexpr int EPI_T = 128;
__global__ void __launch_bounds__(EPI_T)
k_pf_epi(LayerW L, Dims dm, const int32_t* __restrict__ acc, int ld_acc, const int32_t* __restrict__ t, const float* __restrict__ s_x,
         float* __restrict__ zx, int ldz /* row stride of zx: a multiple of 4 floats */)
{
    pdl_wait();
    __shared__ float v_sh[64];
    const int p = blockIdx.y;
    if (threadIdx.x < dm.r) v_sh[threadIdx.x] = fmul(L.in_a_s[threadIdx.x], (float)t[(size_t)p * T_STRIDE + threadIdx.x]);
    __syncthreads();
    const int i = blockIdx.x * EPI_T + threadIdx.x;
    if (i >= dm.d_in_proj) return;
    zx[(size_t)p * ldz + i] = proj_epilogue_row(acc[(size_t)p * ld_acc + i], L.in_row_scale, L.in_B, L.in_b_s, i, dm.r, v_sh, s_x[p]);
}

// the same for lora_rank = 4 * JW: the LoRA sum by lora_up4 (four lanes per row, vector loads of the LoRA-up bytes; k_fin4's scheme)
template <int JW, bool I4 = false>
__global__ void __launch_bounds__(FIN_THREADS)
k_pf_epi4(LayerW L, Dims dm, const int32_t* __restrict__ acc, int ld_acc, const int32_t* __restrict__ t, const float* __restrict__ s_x,
          float* __restrict__ zx, int ldz)
{
    const int p = blockIdx.y, base = blockIdx.x * FIN_THREADS, i = base + threadIdx.x;
    const bool own = i < dm.d_in_proj;
    const int il = own ? i : 0;
    const float rs = __half2float(L.in_row_scale[il]), bs = L.in_b_s[il];      // weights: before pdl_wait
    LoraRegs<JW, I4> lr;
    lora_load4<JW, I4>(L.in_B, L.in_a_s, base, dm.d_in_proj, lr);
    pdl_wait();
    const int acc_i = acc[(size_t)p * ld_acc + il];
    const float sx = s_x[p];
    const double lo = lora_sum4<JW, I4>(lr, t + (size_t)p * T_STRIDE);
    if (own) zx[(size_t)p * ldz + i] = fmul(sx, fadd(fmul(rs, (float)acc_i), fmul(bs, (float)lo)));
}

// S4 for every (position, conv channel) + softplus of dt: the raw samples of positions < 0 come from the sequence's conv ring
// (sample of step tau lives in slot tau mod 4; `ps` = slot of position 0)
constexpr int CONV_T = 256;
__global__ void __launch_bounds__(CONV_T)
k_pf_conv(LayerW L, Dims dm, const float* __restrict__ zx, int ldz, int T, const float* __restrict__ ring /* [conv_dim][4] of the sequence */,
          const int32_t* __restrict__ pos, float* __restrict__ xbc /* [T][conv_dim] */, float* __restrict__ dt /* [T][nheads] */)
{
    pdl_wait();
    const int p = blockIdx.y;
    const int c = blockIdx.x * CONV_T + threadIdx.x;
    const int ps = pos[0] & 3;
    if (c < dm.conv_dim) {
        const float* col = zx + dm.d_inner + c;             // raw x|B|C sample of position q: col[q * ldz]
        float s[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int q = p - 3 + j;
            s[j] = q >= 0 ? col[(size_t)q * ldz] : ring[4 * (size_t)c + ((ps + q) & 3)];
        }
        const float4 cw = *(const float4*)(L.conv_w + 4 * (size_t)c);
        float o = L.conv_b[c];
        o = ffma(cw.x, s[0], o);
        o = ffma(cw.y, s[1], o);
        o = ffma(cw.z, s[2], o);
        o = ffma(cw.w, s[3], o);
        xbc[(size_t)p * dm.conv_dim + c] = siluf(o);
    } else if (c < dm.conv_dim + dm.nheads) {
        const int h = c - dm.conv_dim;
        dt[(size_t)p * dm.nheads + h] = sp_softplusf(fadd(zx[(size_t)p * ldz + dm.d_inner + dm.conv_dim + h], L.dt_bias[h]));
    }
}

// the conv ring after the chunk: the last min(T, 4) raw samples go to their slots (a separate launch: k_pf_conv reads the ring)
__global__ void k_pf_ring(Dims dm, const float* __restrict__ zx, int ldz, int T, float* __restrict__ ring, const int32_t* __restrict__ pos)
{
    pdl_wait();
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= dm.conv_dim) return;
    const int ps = pos[0] & 3;
    for (int q = T > 4 ? T - 4 : 0; q < T; ++q) ring[4 * (size_t)c + ((ps + q) & 3)] = zx[(size_t)q * ldz + dm.d_inner + c];
}

// S5 + S6 gate, serial over the T positions with the state rows in registers: one CTA owns PB (head, p) rows, LANES lanes per row.
// The inputs of TB positions at a time (B', C' of the head's group, x', z of the CTA's rows, dt of the head) are staged in shared
// memory with cp.async, double-buffered, so that the serial loop reads shared memory only; exp(dt A), dt x and silu(z) of a block
// are made by all threads at once before its loop (same operations as k_ssm: the result is bit-identical to the step path).
constexpr int SEQ_T = 256, SEQ_PB = 16, SEQ_LANES = SEQ_T / SEQ_PB, SEQ_NMAX = 16;      // <= 16 state values per lane: d_state <= 256
constexpr int SEQ_TB = 16;                                                             // positions per staged block (SEQ_TB * SEQ_PB == SEQ_T)
__device__ __forceinline__ void cp_async16(void* dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
inline size_t seq_smem(const Dims& d) { return 2 * sizeof(float) * ((size_t)SEQ_TB * (2 * d.d_state + 2 * SEQ_PB) + SEQ_TB) + sizeof(float) * 3 * SEQ_T; }

__device__ __forceinline__ float st_get(const float* p) { return *p; }
__device__ __forceinline__ float st_get(const __half* p) { return __half2float(*p); }
__device__ __forceinline__ void st_put(float* p, float v) { *p = v; }
__device__ __forceinline__ void st_put(__half* p, float v) { *p = __float2half_rn(v); }      // v is already binary16-representable
__device__ __forceinline__ float st_round(float v, const float*) { return v; }
__device__ __forceinline__ float st_round(float v, const __half*) { return __half2float(__float2half_rn(v)); }     // R24: rounded after EVERY step

template <int NPER, typename ST>       // state values per lane = d_state / SEQ_LANES; state type (fp32, or the fp16 format of R24)
__global__ void __launch_bounds__(SEQ_T)
k_pf_ssm(LayerW L, Dims dm, const float* __restrict__ zx, int ldz, const float* __restrict__ xbc, const float* __restrict__ dtv, int T,
         ST* __restrict__ ssm /* [h][p][n] of the sequence */, float* __restrict__ g /* [T][d_inner] */)
{
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int ds = dm.d_state;
    const int stage_f = SEQ_TB * (2 * ds + 2 * SEQ_PB) + SEQ_TB;          // floats per stage: B | C | x | z | dt
    float* st0 = (float*)smem_raw;
    float* s_dA = st0 + 2 * stage_f;                                       // [TB]   exp(dt A)          (padded to SEQ_T floats)
    float* s_dtx = s_dA + SEQ_T;                                           // [TB][PB] dt * x
    float* s_sz = s_dtx + SEQ_T;                                           // [TB][PB] silu(z)
    const int pblocks = dm.headdim / SEQ_PB;
    const int h = blockIdx.x / pblocks, p0 = (blockIdx.x % pblocks) * SEQ_PB;
    const int grp = h / (dm.nheads / dm.ngroups);
    const int tid = threadIdx.x, p = tid / SEQ_LANES, ln = tid % SEQ_LANES;
    const int ch0 = h * dm.headdim + p0, ch = ch0 + p;
    const int gs = dm.ngroups * ds;
    ST* Hr = ssm + (size_t)ch * ds;
    float hreg[NPER];
    constexpr int nper = NPER;                            // contiguous state values of this lane
#pragma unroll
    for (int k = 0; k < NPER; ++k) hreg[k] = st_get(Hr + ln * nper + k);
    pdl_wait();                                           // (the state rows above were written by this kernel of the chunk before, or by a reset)
    const float An = -sp_expf(L.A_log[h]);
    const float Dh = L.D[h];

    auto issue = [&](int blk) {                           // stage the inputs of positions [blk*TB, blk*TB + TB) (clamped to T)
        float* sb = st0 + (blk & 1) * stage_f;
        float* sB = sb, *sC = sb + SEQ_TB * ds, *sX = sC + SEQ_TB * ds, *sZ = sX + SEQ_TB * SEQ_PB, *sD = sZ + SEQ_TB * SEQ_PB;
        const int q0 = blk * SEQ_TB;
        const int nq = min(SEQ_TB, T - q0);
        const int per = ds / 4;                           // 16-byte pieces per position of B (and of C)
        for (int i = tid; i < nq * per; i += SEQ_T) {
            const int q = i / per, k = i - q * per;
            const float* row = xbc + (size_t)(q0 + q) * dm.conv_dim + dm.d_inner + grp * ds;
            cp_async16(sB + q * ds + 4 * k, row + 4 * k);
            cp_async16(sC + q * ds + 4 * k, row + gs + 4 * k);
        }
        for (int i = tid; i < nq * (SEQ_PB / 4); i += SEQ_T) {
            const int q = i / (SEQ_PB / 4), k = i - q * (SEQ_PB / 4);
            cp_async16(sX + q * SEQ_PB + 4 * k, xbc + (size_t)(q0 + q) * dm.conv_dim + ch0 + 4 * k);
            cp_async16(sZ + q * SEQ_PB + 4 * k, zx + (size_t)(q0 + q) * ldz + ch0 + 4 * k);
        }
        if (tid < nq) cp_async4(sD + tid, dtv + (size_t)(q0 + tid) * dm.nheads + h);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    const int nblk = (T + SEQ_TB - 1) / SEQ_TB;
    issue(0);
    for (int blk = 0; blk < nblk; ++blk) {
        if (blk + 1 < nblk) {
            issue(blk + 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
        const float* sb = st0 + (blk & 1) * stage_f;
        const float* sB = sb, *sC = sb + SEQ_TB * ds, *sX = sC + SEQ_TB * ds, *sZ = sX + SEQ_TB * SEQ_PB, *sD = sZ + SEQ_TB * SEQ_PB;
        const int q0 = blk * SEQ_TB;
        const int nq = min(SEQ_TB, T - q0);
        {   // per-block scalars, one (position, row) per thread
            const int q = tid / SEQ_PB, r = tid % SEQ_PB;
            if (q < nq) {
                const float d = sD[q];
                if (r == 0) s_dA[q] = sp_expf(fmul(d, An));
                s_dtx[tid] = fmul(d, sX[tid]);
                s_sz[tid] = siluf(sZ[tid]);
            }
        }
        __syncthreads();
#pragma unroll 4
        for (int q = 0; q < nq; ++q) {
            const float dA = s_dA[q];
            const float dtx = s_dtx[q * SEQ_PB + p];
            const float* Bc = sB + q * ds + ln * nper;
            const float* Cc = sC + q * ds + ln * nper;
            float bv[NPER], cv[NPER];
            if constexpr (NPER % 4 == 0) {
#pragma unroll
                for (int k = 0; k < NPER; k += 4) {
                    const float4 b4 = *(const float4*)(Bc + k), c4 = *(const float4*)(Cc + k);
                    bv[k] = b4.x; bv[k + 1] = b4.y; bv[k + 2] = b4.z; bv[k + 3] = b4.w;
                    cv[k] = c4.x; cv[k + 1] = c4.y; cv[k + 2] = c4.z; cv[k + 3] = c4.w;
                }
            } else {
#pragma unroll
                for (int k = 0; k < NPER; ++k) { bv[k] = Bc[k]; cv[k] = Cc[k]; }
            }
            double a2[2] = { 0.0, 0.0 };                   // two chains (any tree: DESIGN.md 5.3)
#pragma unroll
            for (int k = 0; k < NPER; ++k) {
                const float hn = ffma(dA, hreg[k], fmul(dtx, bv[k]));
                hreg[k] = st_round(hn, Hr);                // what the next position reads
                a2[k & 1] = dacc(a2[k & 1], cv[k], hn);   // the readout of this position uses the unrounded value
            }
            double a = a2[0] + a2[1];
#pragma unroll
            for (int o = SEQ_LANES / 2; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o, SEQ_LANES);
            if (ln == 0) {
                a = dacc(a, Dh, sX[q * SEQ_PB + p]);
                const float y = (float)a;
                g[(size_t)(q0 + q) * dm.d_inner + ch] = fmul(y, s_sz[q * SEQ_PB + p]);
            }
        }
        __syncthreads();                                  // the stage is refilled two blocks on; s_dA / s_dtx / s_sz by the next block
    }
#pragma unroll
    for (int k = 0; k < NPER; ++k) st_put(Hr + ln * nper + k, hreg[k]);
}

// the last position's residual stream becomes the sequence's hidden state
__global__ void k_pf_copy_hidden(const float* __restrict__ u_last, float* __restrict__ u_seq, int d)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < d) u_seq[k] = u_last[k];
}

}  // namespace prefill
}  // namespace dfssm
