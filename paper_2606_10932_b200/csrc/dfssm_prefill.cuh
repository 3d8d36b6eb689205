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
         float* __restrict__ zx)
{
    __shared__ float v_sh[64];
    const int p = blockIdx.y;
    if (threadIdx.x < dm.r) v_sh[threadIdx.x] = fmul(L.in_a_s[threadIdx.x], (float)t[(size_t)p * T_STRIDE + threadIdx.x]);
    __syncthreads();
    const int i = blockIdx.x * EPI_T + threadIdx.x;
    if (i >= dm.d_in_proj) return;
    zx[(size_t)p * dm.d_in_proj + i] = proj_epilogue_row(acc[(size_t)p * ld_acc + i], L.in_row_scale, L.in_B, L.in_b_s, i, dm.r, v_sh, s_x[p]);
}

// S4 for every (position, conv channel) + softplus of dt: the raw samples of positions < 0 come from the sequence's conv ring
// (sample of step tau lives in slot tau mod 4; `ps` = slot of position 0)
constexpr int CONV_T = 256;
__global__ void __launch_bounds__(CONV_T)
k_pf_conv(LayerW L, Dims dm, const float* __restrict__ zx, int T, const float* __restrict__ ring /* [conv_dim][4] of the sequence */,
          const int32_t* __restrict__ pos, float* __restrict__ xbc /* [T][conv_dim] */, float* __restrict__ dt /* [T][nheads] */)
{
    const int p = blockIdx.y;
    const int c = blockIdx.x * CONV_T + threadIdx.x;
    const int ps = pos[0] & 3;
    if (c < dm.conv_dim) {
        const float* col = zx + dm.d_inner + c;             // raw x|B|C sample of position q: col[q * d_in_proj]
        float s[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int q = p - 3 + j;
            s[j] = q >= 0 ? col[(size_t)q * dm.d_in_proj] : ring[4 * (size_t)c + ((ps + q) & 3)];
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
        dt[(size_t)p * dm.nheads + h] = sp_softplusf(fadd(zx[(size_t)p * dm.d_in_proj + dm.d_inner + dm.conv_dim + h], L.dt_bias[h]));
    }
}

// the conv ring after the chunk: the last min(T, 4) raw samples go to their slots (a separate launch: k_pf_conv reads the ring)
__global__ void k_pf_ring(Dims dm, const float* __restrict__ zx, int T, float* __restrict__ ring, const int32_t* __restrict__ pos)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= dm.conv_dim) return;
    const int ps = pos[0] & 3;
    for (int q = T > 4 ? T - 4 : 0; q < T; ++q) ring[4 * (size_t)c + ((ps + q) & 3)] = zx[(size_t)q * dm.d_in_proj + dm.d_inner + c];
}

// S5 + S6 gate, serial over the T positions with the state rows in registers: one CTA owns PB (head, p) rows, LANES lanes per row
constexpr int SEQ_T = 256, SEQ_PB = 16, SEQ_LANES = SEQ_T / SEQ_PB, SEQ_NMAX = 16;      // <= 16 state values per lane: d_state <= 256
__global__ void __launch_bounds__(SEQ_T)
k_pf_ssm(LayerW L, Dims dm, const float* __restrict__ zx, const float* __restrict__ xbc, const float* __restrict__ dtv, int T,
         float* __restrict__ ssm /* [h][p][n] of the sequence */, float* __restrict__ g /* [T][d_inner] */)
{
    const int pblocks = dm.headdim / SEQ_PB;
    const int h = blockIdx.x / pblocks, p0 = (blockIdx.x % pblocks) * SEQ_PB;
    const int grp = h / (dm.nheads / dm.ngroups);
    const int tid = threadIdx.x, p = tid / SEQ_LANES, ln = tid % SEQ_LANES;
    const int ch = h * dm.headdim + p0 + p;
    const int gs = dm.ngroups * dm.d_state;
    float* Hr = ssm + (size_t)ch * dm.d_state;
    float hreg[SEQ_NMAX];
    const int nper = dm.d_state / SEQ_LANES;              // contiguous state values of this lane
#pragma unroll
    for (int k = 0; k < SEQ_NMAX; ++k) hreg[k] = k < nper ? Hr[ln * nper + k] : 0.0f;
    const float An = -sp_expf(L.A_log[h]);
    const float Dh = L.D[h];
    for (int q = 0; q < T; ++q) {
        const float d = dtv[(size_t)q * dm.nheads + h];
        const float dA = sp_expf(fmul(d, An));
        const float* row = xbc + (size_t)q * dm.conv_dim;
        const float xv = row[ch];
        const float dtx = fmul(d, xv);
        const float* Bc = row + dm.d_inner + grp * dm.d_state + ln * nper;
        const float* Cc = row + dm.d_inner + gs + grp * dm.d_state + ln * nper;
        double a = 0.0;
#pragma unroll
        for (int k = 0; k < SEQ_NMAX; ++k) {
            if (k < nper) {
                const float hn = ffma(dA, hreg[k], fmul(dtx, Bc[k]));
                hreg[k] = hn;
                a = dacc(a, Cc[k], hn);
            }
        }
#pragma unroll
        for (int o = SEQ_LANES / 2; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o, SEQ_LANES);
        if (ln == 0) {
            a = dacc(a, Dh, xv);
            const float y = (float)a;
            g[(size_t)q * dm.d_inner + ch] = fmul(y, siluf(zx[(size_t)q * dm.d_in_proj + ch]));
        }
    }
#pragma unroll
    for (int k = 0; k < SEQ_NMAX; ++k)
        if (k < nper) Hr[ln * nper + k] = hreg[k];
}

// the last position's residual stream becomes the sequence's hidden state
__global__ void k_pf_copy_hidden(const float* __restrict__ u_last, float* __restrict__ u_seq, int d)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < d) u_seq[k] = u_last[k];
}

}  // namespace prefill
}  // namespace dfssm
