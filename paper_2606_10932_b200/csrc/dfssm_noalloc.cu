// dfssm_head_noalloc: S8 of the DF-SSM step (final RMSNorm + absmax int8 quantiser, tied int8 LM head, greedy argmax;
// PAPER.md P:96, R16 / R19) as ONE entry point that allocates nothing and needs no context or arena.
//
// Why: some callers cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it) and
// cannot hand the library an arena either.  The intermediates of S8 -- the int8 codes of the normed hidden state, their scale and
// the logits the argmax reads -- live in a file-scope `static __device__` array of DFSSM_NOALLOC_SCRATCH_BYTES (4 MiB), which
// every GPU that loads libdfssm.so holds until the process exits.  The caller passes inputs and outputs only.
//
// The array's name is a host-side stand-in in host code, not a device address: its device address is taken once per device with
// cudaGetSymbolAddress (below, with that device current) and that pointer is what the kernels get.
//
// Sharing: every call on a device uses the same array, and the array keeps the last call's contents.  Nothing in it has to
// start at zero (every value a kernel reads was written by the kernel before it in the same call; the tail beyond a call's need
// is never read), so nothing is cleared.  Calls that OVERLAP on the GPU (two streams, two host threads with different streams,
// graph branches that run side by side) RACE on it: serialise them on one stream or with events.
//
// This file is its own translation unit: it shares dfssm_math.cuh (inline device arithmetic) with the step path and none of its
// kernels, buffers or host code; the arithmetic is the step path's value by value (same rounding points, fp64 sum of squares in
// any tree, exact integers), so logits and tokens are bit-identical to dfssm_step's (tests/test_zz_no_alloc.py).
#include "../../include/dfssm.h"

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "dfssm_math.cuh"

namespace {

using namespace dfssm;

static __device__ __align__(256) unsigned char g_noalloc_scratch[DFSSM_NOALLOC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
unsigned char* g_scratch_dev[MAX_DEVICES];          // device address of g_noalloc_scratch, per device ordinal
bool g_scratch_ready[MAX_DEVICES];
std::mutex g_setup_mutex;
thread_local char g_err[256] = "";

int fail(int code, const char* fmt, ...) __attribute__((format(printf, 2, 3)));
int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }

// set-up, once per device, with that device current
int scratch_for_current_device(unsigned char** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(DFSSM_E_CUDA, "dfssm_head_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(DFSSM_E_ARG, "dfssm_head_noalloc: device ordinal %d beyond %d", dev, MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_ready[dev]) {
        cudaDeviceProp prop;
        e = cudaGetDeviceProperties(&prop, dev);
        if (e != cudaSuccess) return fail(DFSSM_E_CUDA, "dfssm_head_noalloc: cudaGetDeviceProperties: %s", cudaGetErrorString(e));
        if (prop.major != 10) return fail(DFSSM_E_ARCH, "dfssm_head_noalloc: device %d is sm_%d%d, the library is built for sm_100a", dev, prop.major, prop.minor);
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) return fail(DFSSM_E_CUDA, "dfssm_head_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        g_scratch_dev[dev] = (unsigned char*)p;
        g_scratch_ready[dev] = true;
    }
    *out = g_scratch_dev[dev];
    return DFSSM_OK;
}

// ---- S8 first part: RMSNorm statistics + absmax int8 quantiser of one sequence per CTA (R4) ----
//   rstd = 1/sqrt(mean(x^2) + eps) with the sum in binary64;  amax = max |x*w|;  q = rint(x*w * (127/amax));  s = amax*rstd/127
constexpr int NQ_T = 512;
__global__ void __launch_bounds__(NQ_T)
k_na_normquant(const float* __restrict__ hidden, const float* __restrict__ w, int d, float eps,
               int8_t* __restrict__ codes /* [batch][d] */, float* __restrict__ scale /* [batch] */)
{
    __shared__ double sh_d[NQ_T / 32];
    __shared__ float sh_f[NQ_T / 32];
    __shared__ float sh_bcast[2];
    const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const float* x = hidden + (size_t)b * d;
    double ss = 0.0;
    float amax = 0.0f;
    for (int k = tid; k < d; k += NQ_T) {
        const float v = x[k];
        ss = dacc(ss, v, v);
        amax = fmaxf(amax, fabsf(fmul(v, w[k])));
    }
    ss = warp_sum(ss);
    amax = warp_max(amax);
    if (lane == 0) { sh_d[wid] = ss; sh_f[wid] = amax; }
    __syncthreads();
    if (wid == 0) {
        double s2 = lane < NQ_T / 32 ? sh_d[lane] : 0.0;
        float m2 = lane < NQ_T / 32 ? sh_f[lane] : 0.0f;
        s2 = warp_sum(s2);
        m2 = warp_max(m2);
        if (lane == 0) {
            const float ms = (float)(s2 / (double)d);
            sh_bcast[0] = m2;
            sh_bcast[1] = fdiv(1.0f, __fsqrt_rn(fadd(ms, eps)));
        }
    }
    __syncthreads();
    amax = sh_bcast[0];
    const float rstd = sh_bcast[1];
    const float inv = amax == 0.0f ? 0.0f : fdiv(127.0f, amax);
    for (int k = tid; k < d; k += NQ_T) codes[(size_t)b * d + k] = (int8_t)(amax == 0.0f ? 0 : quant_code(fmul(x[k], w[k]), inv));
    if (tid == 0) scale[b] = amax == 0.0f ? 0.0f : fdiv(fmul(amax, rstd), 127.0f);
}

// ---- S8 second part: tied int8 LM head, logit_v = float(sum_k E_vk * q_k) * (s_h * e_s[v])   (R16); one warp per row ----
//   The codes of up to HEAD_BT sequences sit in shared memory; an embedding row is read once for all of them.
constexpr int LM_T = 256, HEAD_BT = 8;
__global__ void __launch_bounds__(LM_T)
k_na_lmhead(const int8_t* __restrict__ E, const float* __restrict__ e_s, int vocab, int K, const int8_t* __restrict__ codes,
            const float* __restrict__ s_h, int batch, float* __restrict__ logits /* scratch [batch][vocab] */,
            float* __restrict__ logits_out /* caller's copy, or null */)
{
    extern __shared__ __align__(16) uint8_t smem[];
    const int b0 = blockIdx.y * HEAD_BT;
    const int nb = min(HEAD_BT, batch - b0);
    int8_t* sq = (int8_t*)smem;
    for (int i = threadIdx.x; i < nb * (K / 16); i += LM_T) ((int4*)sq)[i] = ((const int4*)(codes + (size_t)b0 * K))[i];
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int row = blockIdx.x * (LM_T / 32) + wid; row < vocab; row += gridDim.x * (LM_T / 32)) {
        const int4* erow = (const int4*)(E + (size_t)row * K);
        int s[HEAD_BT];
#pragma unroll
        for (int bb = 0; bb < HEAD_BT; ++bb) s[bb] = 0;
        for (int c = lane; c < K / 16; c += 32) {
            const int4 a4 = __ldg(erow + c);
#pragma unroll
            for (int bb = 0; bb < HEAD_BT; ++bb) {
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
        for (int bb = 0; bb < HEAD_BT; ++bb) {
            if (bb < nb) {
                const int tot = warp_sum_i(s[bb]);
                if (lane == 0) {
                    const float lg = fmul((float)tot, fmul(s_h[b0 + bb], es));
                    logits[(size_t)(b0 + bb) * vocab + row] = lg;
                    if (logits_out) logits_out[(size_t)(b0 + bb) * vocab + row] = lg;
                }
            }
        }
    }
}

// ---- S8 last part: greedy token = argmax, the lowest index on ties (R19); one CTA per sequence ----
constexpr int AM_T = 1024;
__global__ void __launch_bounds__(AM_T)
k_na_argmax(const float* __restrict__ logits, int vocab, int32_t* __restrict__ next)
{
    __shared__ float sv[AM_T / 32];
    __shared__ int si[AM_T / 32];
    const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const float* lg = logits + (size_t)b * vocab;
    float best = -INFINITY;
    int bi = 0x7fffffff;
    for (int i = tid; i < vocab; i += AM_T) {
        const float x = lg[i];
        if (x > best || (x == best && i < bi)) { best = x; bi = i; }
    }
    auto fold = [&]() {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
        }
    };
    fold();
    if (lane == 0) { sv[wid] = best; si[wid] = bi; }
    __syncthreads();
    if (wid == 0) {
        best = sv[lane];
        bi = si[lane];
        fold();
        if (lane == 0) next[b] = bi == 0x7fffffff ? 0 : bi;
    }
}

}  // namespace

extern "C" {

size_t dfssm_head_noalloc_scratch_need(int batch, int d_model, int vocab)
{
    if (batch < 1 || d_model < 1 || vocab < 1) return 0;
    return up256((size_t)batch * d_model) + up256((size_t)batch * 4) + (size_t)batch * vocab * 4;
}

const char* dfssm_head_noalloc_error(void) { return g_err; }

int dfssm_head_noalloc(const float* hidden_dev, const float* normf_w_dev, const int8_t* emb_dev, const float* emb_scale_dev,
                       int batch, int d_model, int vocab, float eps, int32_t* next_dev, float* logits_dev, void* cuda_stream)
{
    g_err[0] = 0;
    if (!hidden_dev || !normf_w_dev || !emb_dev || !emb_scale_dev || !next_dev)
        return fail(DFSSM_E_ARG, "dfssm_head_noalloc: null pointer");
    if (batch < 1 || vocab < 1 || d_model < 16 || d_model % 16 != 0)
        return fail(DFSSM_E_ARG, "dfssm_head_noalloc: batch %d, vocab %d must be >= 1 and d_model %d a positive multiple of 16", batch, vocab, d_model);
    if (((uintptr_t)emb_dev & 15) != 0) return fail(DFSSM_E_ARG, "dfssm_head_noalloc: emb_dev must be 16-byte aligned");
    const size_t need = dfssm_head_noalloc_scratch_need(batch, d_model, vocab);
    if (need > (size_t)DFSSM_NOALLOC_SCRATCH_BYTES)
        return fail(DFSSM_E_SIZE, "dfssm_head_noalloc: batch %d x (d_model %d + vocab %d) needs %zu bytes of scratch, the static array holds %u "
                                  "(DFSSM_NOALLOC_SCRATCH_BYTES): use a smaller batch or the arena path (dfssm_step)",
                    batch, d_model, vocab, need, (unsigned)DFSSM_NOALLOC_SCRATCH_BYTES);
    const size_t lm_smem = (size_t)HEAD_BT * d_model;
    if (lm_smem > 48 * 1024) return fail(DFSSM_E_ARG, "dfssm_head_noalloc: d_model %d beyond %d", d_model, 48 * 1024 / HEAD_BT);
    unsigned char* scratch = nullptr;
    const int rc = scratch_for_current_device(&scratch);
    if (rc != DFSSM_OK) return rc;
    int8_t* codes = (int8_t*)scratch;
    float* scale = (float*)(scratch + up256((size_t)batch * d_model));
    float* logits = (float*)(scratch + up256((size_t)batch * d_model) + up256((size_t)batch * 4));
    cudaStream_t st = (cudaStream_t)cuda_stream;

    k_na_normquant<<<batch, NQ_T, 0, st>>>(hidden_dev, normf_w_dev, d_model, eps, codes, scale);
    const int per = LM_T / 32;
    int gx = (vocab + per - 1) / per;
    if (gx > 148 * 16) gx = 148 * 16;
    k_na_lmhead<<<dim3(gx, (batch + HEAD_BT - 1) / HEAD_BT), LM_T, lm_smem, st>>>(emb_dev, emb_scale_dev, vocab, d_model, codes, scale, batch,
                                                                                  logits, logits_dev);
    k_na_argmax<<<batch, AM_T, 0, st>>>(logits, vocab, next_dev);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DFSSM_E_CUDA, "dfssm_head_noalloc: launch: %s", cudaGetErrorString(e));
    return DFSSM_OK;
}

}  // extern "C"
