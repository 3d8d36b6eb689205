// Host side of libdfssm.so: the C ABI of include/dfssm.h.
// Arena carving, canonical-blob parsing (this is the CUDA path's own parser),
// the kernel chain of one decode step and its CUDA-graph launcher ("CUDA graph capture ...
// primary source of the large batch=1 speedup").
#include "../../include/dfssm.h"

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "dfssm_kernels.cuh"
#include "dfssm_mega_host.cuh"
#include "dfssm_mma.cuh"
#include "dfssm_prefill.cuh"

using namespace dfssm;

namespace {

constexpr size_t ARENA_ALIGN = 256;
inline size_t up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Carve {                 // byte offsets inside the arena
    size_t blob, ssm, conv, pos, u, xq, xqp, sx, qsum, acc, t, g, bcdt, logits, next, tok, err, taps, total;
    size_t p_tok, p_u, p_xq, p_xqp, p_sx, p_qsum, p_acc, p_t, p_zx, p_xbc, p_dt, p_g;      // prefill: activations of one chunk of positions
    size_t m_chunks, m_schunks, m_blocks, m_x, m_xbytes, m_am, m_prof;      // mega path regions (valid if mega_fit)
    bool mega_fit;
    size_t ssm_elems, ssm_esize, ldq, ld_acc;      // ssm_esize: bytes per state value (4, or 2 with DFSSM_FLAG_STATE_FP16)
    uint32_t tap_stride;
    TapLayout tl;
};

struct GraphEntry { int batch; cudaGraphExec_t exec; };

}  // namespace

struct dfssm_ctx {
    dfssm_config cfg;
    Dims dm;
    Carve cv;
    uint8_t* arena;
    cudaStream_t stream;
    bool loaded;
    bool failed;               // a step timed out on the device: state and exchange records are half-written until dfssm_reset_state(-1)
    size_t blob_bytes;
    std::vector<LayerW> layers;
    const int8_t* emb; const float* emb_s; const float* normf_w;
    std::vector<GraphEntry> graphs;
    int last_batch;
    mega::Params mp;           // layout + pointers of the mega path (batch 1)
    mega::KernelFn mega_fn;    // the instantiation of the persistent kernel that serves this shape
    bool mega_ok;              // the device can co-schedule the mega grid and the shape fits
    uint64_t epoch;            // steps taken by the mega path: makes every exchange flag unique
    int32_t* pinned_tok;       // page-locked staging for dfssm_step_host
    int* pinned_err;
    char err[512];
};

namespace {

int fail(dfssm_ctx* c, int code, const char* fmt, ...)
{
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof c->err, fmt, ap);
        va_end(ap);
    }
    return code;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(ctx, DFSSM_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_));        \
    } while (0)

bool valid_cfg(const dfssm_config* c)
{
    if (!c || c->abi_version != DFSSM_ABI_VERSION) return false;
    if (c->n_layers < 0 || c->d_model <= 0 || c->d_inner <= 0 || c->headdim <= 0 || c->d_state <= 0 ||
        c->ngroups <= 0 || c->vocab <= 0)
        return false;
    if (c->d_conv != 4) return false;
    if (c->d_model % 32 || c->d_inner % 32 || c->d_model > 8192 || c->d_inner > 8192) return false;
    if (c->d_inner % c->headdim || c->headdim % SSM_PB || c->d_state % 4) return false;
    if ((c->d_inner / c->headdim) % c->ngroups) return false;
    if (c->lora_rank < 1 || c->lora_rank > 64) return false;
    if (c->max_batch < 1 || c->max_batch > 256) return false;
    if (!(c->norm_eps > 0.0f)) return false;
    if (c->flags & (DFSSM_FLAG_SCAFFOLD17 | DFSSM_FLAG_LORA_INT4)) {       // format variants: tensor-core projections only
        if (c->d_model % 128 || c->d_inner % 128 || (c->flags & DFSSM_FLAG_NO_MMA)) return false;
        if (c->lora_rank != 8 && c->lora_rank != 16 && c->lora_rank != 32 && c->lora_rank != 64) return false;
    }
    return true;
}

Dims make_dims(const dfssm_config& c)
{
    Dims d;
    d.n_layers = c.n_layers; d.d_model = c.d_model; d.d_inner = c.d_inner; d.headdim = c.headdim;
    d.d_state = c.d_state; d.ngroups = c.ngroups; d.vocab = c.vocab; d.r = c.lora_rank;
    d.nheads = c.d_inner / c.headdim;
    d.d_in_proj = 2 * c.d_inner + 2 * c.ngroups * c.d_state + d.nheads;
    d.conv_dim = c.d_inner + 2 * c.ngroups * c.d_state;
    d.eps = c.norm_eps;
    d.fmt = ((c.flags & DFSSM_FLAG_SCAFFOLD17) ? 1 : 0) | ((c.flags & DFSSM_FLAG_LORA_INT4) ? 2 : 0);
    return d;
}

// canonical blob: 256-byte header, tensors in fixed order, 64-byte aligned
struct BlobWalk {
    size_t off = 256;
    size_t take(size_t bytes) { off = up(off, 64); size_t o = off; off += bytes; return o; }
};

size_t blob_bytes_for(const Dims& d)
{
    BlobWalk w;
    const size_t dm = d.d_model, di = d.d_inner, dip = d.d_in_proj, r = d.r, cd = d.conv_dim, nh = d.nheads;
    const size_t pl = (d.fmt & 1) ? 5 : 1, ld = (d.fmt & 2) ? 2 : 1;      // bit planes per sign word; LoRA values per byte
    for (int l = 0; l < d.n_layers; ++l) {
        w.take(4 * dm); w.take(4 * dip * (dm / 32) * pl); w.take(2 * dip); w.take(r * dm / ld); w.take(4 * r);
        w.take(dip * r / ld); w.take(4 * dip); w.take(16 * cd); w.take(4 * cd); w.take(4 * nh); w.take(4 * nh);
        w.take(4 * nh); w.take(4 * di); w.take(4 * dm * (di / 32) * pl); w.take(2 * dm); w.take(r * di / ld);
        w.take(4 * r); w.take(dm * r / ld); w.take(4 * dm);
    }
    w.take((size_t)d.vocab * dm); w.take(4 * (size_t)d.vocab); w.take(4 * dm);
    return up(w.off, 64);
}

Carve carve(const dfssm_config& c)
{
    const Dims d = make_dims(c);
    Carve v;
    memset(&v, 0, sizeof v);
    const size_t B = c.max_batch, nl = c.n_layers > 0 ? c.n_layers : 1;
    v.ssm_elems = (size_t)d.nheads * d.headdim * d.d_state;
    v.ldq = up((size_t)(d.d_model > d.d_inner ? d.d_model : d.d_inner), 64);
    v.ld_acc = up((size_t)(d.d_in_proj > d.d_model ? d.d_in_proj : d.d_model), 4);
    size_t o = 0;
    auto put = [&](size_t bytes) { o = up(o, ARENA_ALIGN); size_t at = o; o += bytes; return at; };
    v.blob = put(blob_bytes_for(d));
    v.ssm_esize = (c.flags & DFSSM_FLAG_STATE_FP16) ? 2 : 4;
    v.ssm = put(nl * B * v.ssm_elems * v.ssm_esize);
    v.conv = put(nl * B * (size_t)d.conv_dim * 16);
    v.pos = put(B * 4);
    v.u = put(B * d.d_model * 4);
    v.xq = put(B * v.ldq);
    v.xqp = put(B * v.ldq);
    v.sx = put(B * 4);
    v.qsum = put(B * 4);
    v.acc = put(B * v.ld_acc * 4);
    v.t = put(B * T_STRIDE * 4);
    v.g = put(B * d.d_inner * 4);
    v.bcdt = put(B * (size_t)(d.d_in_proj + d.nheads) * 4);      // k_fin's finished in_proj values (fin)
    v.logits = put(B * (size_t)d.vocab * 4);
    v.next = put(B * 4);
    v.tok = put(B * 4);
    v.err = put(16);
    {
        const size_t C = prefill::CHUNK;
        v.p_tok = put(C * 4); v.p_u = put(C * d.d_model * 4); v.p_xq = put(C * v.ldq); v.p_xqp = put(C * v.ldq); v.p_sx = put(C * 4);
        v.p_qsum = put(C * 4); v.p_acc = put(C * v.ld_acc * 4); v.p_t = put(C * T_STRIDE * 4); v.p_zx = put(C * v.ld_acc * 4);
        v.p_xbc = put(C * (size_t)d.conv_dim * 4); v.p_dt = put(C * (size_t)d.nheads * 4); v.p_g = put(C * d.d_inner * 4);
    }
    const size_t sizes[DFSSM_TAP_COUNT] = {
        (size_t)d.d_model, 4, 4 * (size_t)d.d_in_proj, 4 * (size_t)d.r, 4 * (size_t)d.d_in_proj,
        4 * (size_t)d.conv_dim, 4 * (size_t)d.nheads, 4 * (size_t)d.d_inner, 4 * (size_t)d.d_inner,
        (size_t)d.d_inner, 4, 4 * (size_t)d.d_model, 4 * (size_t)d.r, 4 * (size_t)d.d_model };
    size_t to = 0;
    for (int i = 0; i < DFSSM_TAP_COUNT; ++i) { v.tl.off[i] = (uint32_t)to; to = up(to + sizes[i], 64); }
    v.tl.off[DFSSM_TAP_COUNT] = (uint32_t)to;
    v.tap_stride = (uint32_t)to;
    v.taps = (c.flags & DFSSM_FLAG_TAPS) ? put(nl * B * to) : 0;
    mega::Params mp;
    v.mega_fit = !(c.flags & (DFSSM_FLAG_NO_MEGA | DFSSM_FLAG_STATE_FP16)) && d.fmt == 0 && mega::plan(d, mega::GRID, mp);      // the persistent kernel keeps fp32 state
    if (v.mega_fit) {
        const mega::Regions rg = mega::regions(mp);
        v.m_chunks = put(rg.chunks);
        v.m_schunks = put(rg.schunks);
        v.m_blocks = put(rg.blocks);
        v.m_x = put(rg.xbuf);
        v.m_xbytes = rg.xbuf;
        v.m_am = put(rg.am);
        v.m_prof = (c.flags & DFSSM_FLAG_PROF) ? put((size_t)mp.G * (mp.L + 1) * mega::PROF_NPH * 8) : 0;
    }
    v.total = up(o, ARENA_ALIGN);
    return v;
}

size_t tap_bytes(const Dims& d, int which)
{
    switch (which) {
        case DFSSM_TAP_XQ_IN: return d.d_model;
        case DFSSM_TAP_S_IN: case DFSSM_TAP_S_G: return 4;
        case DFSSM_TAP_ACC_IN: case DFSSM_TAP_ZXBCDT: return 4 * (size_t)d.d_in_proj;
        case DFSSM_TAP_T_IN: case DFSSM_TAP_T_OUT: return 4 * (size_t)d.r;
        case DFSSM_TAP_XBC_CONV: return 4 * (size_t)d.conv_dim;
        case DFSSM_TAP_DT: return 4 * (size_t)d.nheads;
        case DFSSM_TAP_Y: case DFSSM_TAP_G: return 4 * (size_t)d.d_inner;
        case DFSSM_TAP_GQ: return d.d_inner;
        case DFSSM_TAP_ACC_OUT: case DFSSM_TAP_HIDDEN: return 4 * (size_t)d.d_model;
    }
    return 0;
}

template <typename T> T* at(dfssm_ctx* c, size_t off) { return reinterpret_cast<T*>(c->arena + off); }

}  // namespace

// =================================================================================================
// the kernel chain of one step
// =================================================================================================
namespace {

struct KTimer {                       // optional per-kernel-class device timing (dfssm_time_kernels)
    std::vector<cudaEvent_t> ev;
    std::vector<int> cls;
    cudaStream_t st;
    bool on = false;
    void begin(int k)
    {
        if (!on) return;
        cudaEvent_t a, b;
        cudaEventCreate(&a); cudaEventCreate(&b);
        cudaEventRecord(a, st);
        ev.push_back(a); ev.push_back(b); cls.push_back(k);
    }
    void end()
    {
        if (!on) return;
        cudaEventRecord(ev.back(), st);
    }
};

size_t proj_smem(int K) { return (size_t)PROJ_BT * 2 * K; }
size_t lm_smem(int K) { return (size_t)PROJ_BT * K; }

int proj_grid(int rows_total)
{
    const int per = PROJ_THREADS / 32;
    int g = (rows_total + per - 1) / per;
    const int cap = 148 * 8;
    return g < cap ? g : cap;
}

// the projections run on the tensor cores (tcgen05 kind::i8 on +-1 tiles unpacked in shared memory) from this batch size on
bool use_mma(const dfssm_ctx* c, int batch, int K)
{
    // measured (ms/step, dp4a rows / tensor cores, final build with k_epi_norm4 on the tensor-core chain): cfg 3 batch 4 1.63 / 1.20;
    // cfg 1 (d_model 768) batch 2 0.413 / 0.406, 3 0.458 / 0.424, 5 0.492 / 0.453, 7 0.541 / 0.482; cfg 0 (d_model 256) batch 2
    // 0.037 / 0.041, 4 0.040 / 0.043, 7 0.044 / 0.046, 8 0.046 / 0.046: from batch 4 on for the wide models (up to 3 the persistent
    // kernel serves them), from 2 on for d_model 512 .. 1023, from 8 on below
    if (c->dm.fmt) return true;                       // the format variants are unpacked by k_proj_mma only
    static const int mma_env = getenv("DFSSM_MMA_MIN") ? atoi(getenv("DFSSM_MMA_MIN")) : 0;      // measurement switch
    const int mma_min = mma_env > 0 ? mma_env : c->dm.d_model >= 1024 ? 4 : c->dm.d_model >= 512 ? 2 : 8;
    return batch >= mma_min && K % mma::KMULT == 0 && !(c->cfg.flags & DFSSM_FLAG_NO_MMA);
}

// one projection on the tensor cores; K is split over CTAs until the grid fills the 148 SMs (partial sums are added
// with integer atomics into zeroed buffers: exact, order-independent)
// K is split until this many CTAs share an SM: a CTA is 4 warps that unpack, issue and wait in turn, so co-resident CTAs are
// what hides its latencies (measured, cfg 3, ms/step at batch 64 / 16: 1 CTA 5.72 / 3.52, 2 CTAs 5.46 / 3.24, 3 CTAs 5.49 / 3.29,
// 4 CTAs 5.53 / 3.23)
constexpr int MMA_CTAS_PER_SM = 2;
// Launch with (PDL_ true) or without the programmatic-stream-serialization attribute: with it the kernel may be scheduled while the
// kernel in front of it in the stream drains; it runs its independent prologue and blocks in pdl_wait() until that kernel has
// completed.  KERNEL_ in parentheses if it has template commas.
#define DFSSM_LAUNCH_EX(PDL_, KERNEL_, GRID_, BLOCK_, SMEM_, ST_, ...)                                \
    do {                                                                                              \
        cudaLaunchConfig_t cfg_ = {};                                                                 \
        cfg_.gridDim = GRID_;                                                                         \
        cfg_.blockDim = BLOCK_;                                                                       \
        cfg_.dynamicSmemBytes = SMEM_;                                                                \
        cfg_.stream = ST_;                                                                            \
        cudaLaunchAttribute at_[1];                                                                   \
        at_[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                               \
        at_[0].val.programmaticStreamSerializationAllowed = 1;                                        \
        cfg_.attrs = at_;                                                                             \
        cfg_.numAttrs = (PDL_) ? 1 : 0;                                                               \
        cudaLaunchKernelEx(&cfg_, KERNEL_, __VA_ARGS__);                                              \
    } while (0)
// k_proj_mma<FMT> for the weight format of the model (the LM head always runs FMT = 0: the embedding is int8 in every format)
#define DFSSM_MMA_LAUNCH(PDL_, FMT_, GRID_, ST_, ...)                                                                        \
    do {                                                                                                               \
        switch (FMT_) {                                                                                                \
            case 1: DFSSM_LAUNCH_EX(PDL_, mma::k_proj_mma<1>, GRID_, mma::THREADS, mma::SMEM_BYTES, ST_, __VA_ARGS__); break;             \
            case 2: DFSSM_LAUNCH_EX(PDL_, mma::k_proj_mma<2>, GRID_, mma::THREADS, mma::SMEM_BYTES, ST_, __VA_ARGS__); break;             \
            case 3: DFSSM_LAUNCH_EX(PDL_, mma::k_proj_mma<3>, GRID_, mma::THREADS, mma::SMEM_BYTES, ST_, __VA_ARGS__); break;             \
            default: DFSSM_LAUNCH_EX(PDL_, mma::k_proj_mma<0>, GRID_, mma::THREADS, mma::SMEM_BYTES, ST_, __VA_ARGS__); break;            \
        }                                                                                                              \
    } while (0)
int launch_proj_mma(dfssm_ctx* ctx, const uint32_t* sign, const int8_t* A, int rows, int K, int batch, bool pdl)
{
    const Dims& d = ctx->dm;
    const Carve& v = ctx->cv;
    const int mt = (rows + d.r + mma::TM - 1) / mma::TM, nt = (batch + mma::TN - 1) / mma::TN, nchunk = (K + mma::KC - 1) / mma::KC;
    static const int cps = getenv("DFSSM_MMA_CPS") ? atoi(getenv("DFSSM_MMA_CPS")) : MMA_CTAS_PER_SM;
    int ks = (148 * cps) / (mt * nt);
    if (ks < 1) ks = 1;
    if (ks > nchunk) ks = nchunk;
    int32_t* acc = at<int32_t>(ctx, v.acc);
    int32_t* t = at<int32_t>(ctx, v.t);
    // ks > 1: acc / t were zeroed by the k_normquant launch in front of this projection
    DFSSM_MMA_LAUNCH(pdl, d.fmt, dim3(mt, nt, ks), ctx->stream, sign, A, rows, d.r, K, at<int8_t>(ctx, v.xq), (int)v.ldq, batch, acc, (int)v.ld_acc, t,
                     at<int>(ctx, v.err), nullptr, nullptr, nullptr);
    return DFSSM_OK;
}

// threads per CTA of k_epi_norm4 (S7 + the norm / quantiser behind it in one cluster launch), 0 = this shape runs them apart
int epi_norm_threads(const Dims& d)
{
    if (d.r != 8 && d.r != 16 && d.r != 32 && d.r != 64) return 0;
    if (d.d_model % 256 == 0 && d.d_model / 256 <= 8) return 256;
    if (d.d_model % 512 == 0 && d.d_model / 512 <= 8) return 512;
    return 0;
}
#define DFSSM_LAUNCH_CL(PDL_, KERNEL_, GRID_, BLOCK_, ST_, ...)                                       \
    do {                                                                                              \
        cudaLaunchConfig_t cfg_ = {};                                                                 \
        cfg_.gridDim = GRID_;                                                                         \
        cfg_.blockDim = BLOCK_;                                                                       \
        cfg_.stream = ST_;                                                                            \
        cudaLaunchAttribute at_[2];                                                                   \
        at_[0].id = cudaLaunchAttributeClusterDimension;                                              \
        at_[0].val.clusterDim.x = (GRID_).x;                                                          \
        at_[0].val.clusterDim.y = 1;                                                                  \
        at_[0].val.clusterDim.z = 1;                                                                  \
        at_[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;                               \
        at_[1].val.programmaticStreamSerializationAllowed = 1;                                        \
        cfg_.attrs = at_;                                                                             \
        cfg_.numAttrs = (PDL_) ? 2 : 1;                                                               \
        cudaLaunchKernelEx(&cfg_, KERNEL_, __VA_ARGS__);                                              \
    } while (0)
void launch_epi_norm(const LayerW& L, const Dims& d, int n, const int32_t* acc, int ld_acc, const int32_t* t, const float* s_g, float* u,
                     const float* w_next, int8_t* xq, int ldq, float* s_out, int32_t* zero_acc, int32_t* zero_t, cudaStream_t st, bool pdl)
{
    const int nthr = epi_norm_threads(d);
    const dim3 g(d.d_model / nthr, n);
    const bool i4 = (d.fmt & 2) != 0;
#define DFSSM_EPN_ARGS L, d.d_model, acc, ld_acc, t, s_g, u, w_next, d.eps, xq, ldq, s_out, zero_acc, zero_t
    switch (d.r) {
        case 8:
            if (i4) DFSSM_LAUNCH_CL(pdl, (k_epi_norm4<2, true>), g, nthr, st, DFSSM_EPN_ARGS);
            else DFSSM_LAUNCH_CL(pdl, (k_epi_norm4<2, false>), g, nthr, st, DFSSM_EPN_ARGS);
            break;
        case 16:
            if (i4) DFSSM_LAUNCH_CL(pdl, (k_epi_norm4<4, true>), g, nthr, st, DFSSM_EPN_ARGS);
            else DFSSM_LAUNCH_CL(pdl, (k_epi_norm4<4, false>), g, nthr, st, DFSSM_EPN_ARGS);
            break;
        case 32:
            if (i4) DFSSM_LAUNCH_CL(pdl, (k_epi_norm4<8, true>), g, nthr, st, DFSSM_EPN_ARGS);
            else DFSSM_LAUNCH_CL(pdl, (k_epi_norm4<8, false>), g, nthr, st, DFSSM_EPN_ARGS);
            break;
        default:
            if (i4) DFSSM_LAUNCH_CL(pdl, (k_epi_norm4<16, true>), g, nthr, st, DFSSM_EPN_ARGS);
            else DFSSM_LAUNCH_CL(pdl, (k_epi_norm4<16, false>), g, nthr, st, DFSSM_EPN_ARGS);
            break;
    }
#undef DFSSM_EPN_ARGS
}

// S7 epilogue + residual for n sequences / positions: four lanes per row when the LoRA rank allows (k_epi_out4)
void launch_epi_out(const LayerW& L, const Dims& d, int n, const int32_t* acc, int ld_acc, const int32_t* t, const float* s_g, float* u,
                    uint8_t* tp, uint32_t tap_stride, uint32_t tap_off, cudaStream_t st, bool pdl = false)
{
    const dim3 g4((d.d_model + FIN_THREADS - 1) / FIN_THREADS, n);
    const bool i4 = (d.fmt & 2) != 0;
    switch (d.r) {
        case 8:
            if (i4) DFSSM_LAUNCH_EX(pdl, (k_epi_out4<2, true>), g4, FIN_THREADS, 0, st, L, d.d_model, acc, ld_acc, t, s_g, u, tp, tap_stride, tap_off);
            else DFSSM_LAUNCH_EX(pdl, (k_epi_out4<2, false>), g4, FIN_THREADS, 0, st, L, d.d_model, acc, ld_acc, t, s_g, u, tp, tap_stride, tap_off);
            break;
        case 16:
            if (i4) DFSSM_LAUNCH_EX(pdl, (k_epi_out4<4, true>), g4, FIN_THREADS, 0, st, L, d.d_model, acc, ld_acc, t, s_g, u, tp, tap_stride, tap_off);
            else DFSSM_LAUNCH_EX(pdl, (k_epi_out4<4, false>), g4, FIN_THREADS, 0, st, L, d.d_model, acc, ld_acc, t, s_g, u, tp, tap_stride, tap_off);
            break;
        case 32:
            if (i4) DFSSM_LAUNCH_EX(pdl, (k_epi_out4<8, true>), g4, FIN_THREADS, 0, st, L, d.d_model, acc, ld_acc, t, s_g, u, tp, tap_stride, tap_off);
            else DFSSM_LAUNCH_EX(pdl, (k_epi_out4<8, false>), g4, FIN_THREADS, 0, st, L, d.d_model, acc, ld_acc, t, s_g, u, tp, tap_stride, tap_off);
            break;
        case 64:
            if (i4) DFSSM_LAUNCH_EX(pdl, (k_epi_out4<16, true>), g4, FIN_THREADS, 0, st, L, d.d_model, acc, ld_acc, t, s_g, u, tp, tap_stride, tap_off);
            else DFSSM_LAUNCH_EX(pdl, (k_epi_out4<16, false>), g4, FIN_THREADS, 0, st, L, d.d_model, acc, ld_acc, t, s_g, u, tp, tap_stride, tap_off);
            break;
        default:
            k_epi_out<<<dim3((d.d_model + EPI_THREADS - 1) / EPI_THREADS, n), EPI_THREADS, 0, st>>>(L, d.d_model, d.r, acc, ld_acc, t, s_g, u, tp, tap_stride,
                                                                                                  tap_off);
    }
}

// S7 + the norm / quantiser behind it as one cluster launch (k_epi_norm4): tensor-core chain with dependent launches, no taps
bool fused_epi_norm(const dfssm_ctx* c, int batch)
{
    static const int fuse_env = getenv("DFSSM_FUSE_EPI") ? atoi(getenv("DFSSM_FUSE_EPI")) : 1;
    static const int pdl_env = getenv("DFSSM_PDL_MASK") ? atoi(getenv("DFSSM_PDL_MASK")) : -1;
    if (!fuse_env || pdl_env == 0 || (c->cfg.flags & DFSSM_FLAG_TAPS)) return false;
    return use_mma(c, batch, c->dm.d_model) && use_mma(c, batch, c->dm.d_inner) && epi_norm_threads(c->dm) != 0;
}

// Enqueue S0, L x (S1..S7), S8 for `batch` sequences on the context's stream.  The input tokens are
// read from the arena's own token buffer (cv.tok), which the argmax kernel also refreshes with the
// greedy tokens -- so a graph captured once per batch size serves every caller pointer.
int enqueue_step(dfssm_ctx* c, int batch, KTimer* tm, int* n_launch)
{
    dfssm_ctx* ctx = c;
    const Dims& d = c->dm;
    const Carve& v = c->cv;
    cudaStream_t st = c->stream;
    const size_t B = c->cfg.max_batch;
    KTimer dummy;
    if (!tm) tm = &dummy;
    int nl = 0;

    float* u = at<float>(c, v.u);
    int8_t* xq = at<int8_t>(c, v.xq);
    int8_t* xqp = at<int8_t>(c, v.xqp);
    float* sx = at<float>(c, v.sx);
    int32_t* qsum = at<int32_t>(c, v.qsum);
    int32_t* acc = at<int32_t>(c, v.acc);
    int32_t* t = at<int32_t>(c, v.t);
    float* g = at<float>(c, v.g);
    float* logits = at<float>(c, v.logits);
    int32_t* next = at<int32_t>(c, v.next);
    int32_t* tokens = at<int32_t>(c, v.tok);
    int32_t* pos = at<int32_t>(c, v.pos);
    int* err = at<int>(c, v.err);
    const bool taps_on = (c->cfg.flags & DFSSM_FLAG_TAPS) != 0;
    const int ldq = (int)v.ldq, ld_acc = (int)v.ld_acc;
    // programmatic dependent launch, per kind of kernel (bit set = that kernel may start under the one in front of it):
    // 1 k_normquant(u), 2 in_proj, 4 k_fin4, 8 k_ssm_stream, 16 k_normquant(g), 32 out_proj, 64 k_epi_out4.  Tensor-core chain only.
    // Measured (cfg 3, ms/step without / with, final build): batch 5 1.78 / 1.36, 8 1.90 / 1.53, 16 2.20 / 1.85, 32 2.72 / 2.53,
    // 64 3.99 / 3.80; cfg 4 batch 8 3.02 / 2.53.  DFSSM_PDL_MASK in the environment overrides the choice (0 = off).
    const bool mma_in = use_mma(c, batch, d.d_model), mma_out = use_mma(c, batch, d.d_inner);      // K = d_model: in_proj and the LM head
    static const int pdl_env = getenv("DFSSM_PDL_MASK") ? atoi(getenv("DFSSM_PDL_MASK")) : -1;
    const int pdl = (tm == &dummy && !taps_on) ? (pdl_env >= 0 ? pdl_env : 127) : 0;

    const bool fuse = pdl && fused_epi_norm(c, batch);

    tm->begin(DFSSM_KCLASS_EMBED);
    k_embed<<<dim3((d.d_model + 255) / 256, batch), 256, 0, st>>>(tokens, c->emb, c->emb_s, d.vocab, d.d_model, u, err);
    tm->end(); ++nl;

    for (int l = 0; l < d.n_layers; ++l) {
        const LayerW& L = c->layers[l];
        uint8_t* tp = taps_on ? at<uint8_t>(c, v.taps) + (size_t)l * B * v.tap_stride : nullptr;
        uint8_t* ssm_b = c->arena + v.ssm + (size_t)l * B * v.ssm_elems * v.ssm_esize;
        float* ssm = (float*)ssm_b;
        __half* ssm_h = (__half*)ssm_b;
        const bool st16 = v.ssm_esize == 2;
        float* conv = at<float>(c, v.conv) + (size_t)l * B * (size_t)d.conv_dim * 4;

        tm->begin(DFSSM_KCLASS_NORMQUANT);
        if (!fuse || l == 0)
        DFSSM_LAUNCH_EX(pdl & 1, k_normquant, batch, NQ_THREADS, 0, st, u, d.d_model, L.norm_w, d.d_model, d.eps, xq, mma_in ? nullptr : xqp, ldq, sx,
                        mma_in ? nullptr : qsum,
                        tp, v.tap_stride, v.tl.off[DFSSM_TAP_XQ_IN], v.tl.off[DFSSM_TAP_S_IN],
                        use_mma(c, batch, d.d_model) ? acc : nullptr, (int)ld_acc, t);
        tm->end(); ++nl;

        tm->begin(DFSSM_KCLASS_PROJ_IN);
        if (use_mma(c, batch, d.d_model)) {
            const int rc = launch_proj_mma(c, L.in_sign, L.in_A, d.d_in_proj, d.d_model, batch, (pdl & 2) != 0);
            if (rc != DFSSM_OK) return rc;
        } else
        DFSSM_LAUNCH_EX(pdl & 2, k_proj, dim3(proj_grid(d.d_in_proj + d.r), (batch + PROJ_BT - 1) / PROJ_BT), PROJ_THREADS, proj_smem(d.d_model), st,
                        L.in_sign, L.in_A, d.d_in_proj, d.r, d.d_model, xq, xqp, ldq, qsum, batch, acc, ld_acc, t);
        tm->end(); ++nl;
        if (tp) {
            k_tap_copy_i32<<<dim3((d.d_in_proj + 255) / 256, batch), 256, 0, st>>>(acc, ld_acc, d.d_in_proj, tp,
                                                                                  v.tap_stride, v.tl.off[DFSSM_TAP_ACC_IN]);
            k_tap_copy_i32<<<dim3(1, batch), 64, 0, st>>>(t, T_STRIDE, d.r, tp, v.tap_stride, v.tl.off[DFSSM_TAP_T_IN]);
            nl += 2;
        }

        tm->begin(DFSSM_KCLASS_SSM);
        {
        float* fin = at<float>(c, v.bcdt);
        {
            const dim3 gf((d.d_in_proj + FIN_THREADS - 1) / FIN_THREADS, batch);
#define DFSSM_FIN_ARGS L, d, acc, ld_acc, t, sx, conv, pos, fin, tp, v.tap_stride, v.tl
            switch (d.r) {
                case 8:
                    if (d.fmt & 2) DFSSM_LAUNCH_EX(pdl & 4, (k_fin4<2, true>), gf, FIN_THREADS, 0, st, DFSSM_FIN_ARGS);
                    else DFSSM_LAUNCH_EX(pdl & 4, (k_fin4<2, false>), gf, FIN_THREADS, 0, st, DFSSM_FIN_ARGS);
                    break;
                case 16:
                    if (d.fmt & 2) DFSSM_LAUNCH_EX(pdl & 4, (k_fin4<4, true>), gf, FIN_THREADS, 0, st, DFSSM_FIN_ARGS);
                    else DFSSM_LAUNCH_EX(pdl & 4, (k_fin4<4, false>), gf, FIN_THREADS, 0, st, DFSSM_FIN_ARGS);
                    break;
                case 32:
                    if (d.fmt & 2) DFSSM_LAUNCH_EX(pdl & 4, (k_fin4<8, true>), gf, FIN_THREADS, 0, st, DFSSM_FIN_ARGS);
                    else DFSSM_LAUNCH_EX(pdl & 4, (k_fin4<8, false>), gf, FIN_THREADS, 0, st, DFSSM_FIN_ARGS);
                    break;
                case 64:
                    if (d.fmt & 2) DFSSM_LAUNCH_EX(pdl & 4, (k_fin4<16, true>), gf, FIN_THREADS, 0, st, DFSSM_FIN_ARGS);
                    else DFSSM_LAUNCH_EX(pdl & 4, (k_fin4<16, false>), gf, FIN_THREADS, 0, st, DFSSM_FIN_ARGS);
                    break;
                default: k_fin<<<gf, FIN_THREADS, 0, st>>>(DFSSM_FIN_ARGS); break;
            }
#undef DFSSM_FIN_ARGS
        }
        ++nl;
        {
            const dim3 g32(d.headdim / 32, d.nheads, batch), g16(d.headdim / 16, d.nheads, batch);
            const size_t sm = 2 * (size_t)d.d_state * sizeof(float);
#define DFSSM_SSM_GO(PB_, DS_, G_)                                                                                          \
    if (st16) DFSSM_LAUNCH_EX(pdl & 8, (k_ssm_stream<PB_, DS_, __half>), G_, SSM_THREADS, sm, st, L, d, fin, ssm_h, g, tp, v.tap_stride, v.tl);    \
    else DFSSM_LAUNCH_EX(pdl & 8, (k_ssm_stream<PB_, DS_, float>), G_, SSM_THREADS, sm, st, L, d, fin, ssm, g, tp, v.tap_stride, v.tl)
            if (d.headdim % 32 == 0) {
                if (d.d_state == 128) { DFSSM_SSM_GO(32, 128, g32); }
                else if (d.d_state == 64) { DFSSM_SSM_GO(32, 64, g32); }
                else { DFSSM_SSM_GO(32, 0, g32); }
            } else { DFSSM_SSM_GO(16, 0, g16); }
#undef DFSSM_SSM_GO
        }
        }
        tm->end(); ++nl;

        tm->begin(DFSSM_KCLASS_NORMQUANT);
        DFSSM_LAUNCH_EX(pdl & 16, k_normquant, batch, NQ_THREADS, 0, st, g, d.d_inner, L.gnorm_w, d.d_inner, d.eps, xq, mma_out ? nullptr : xqp, ldq, sx,
                        mma_out ? nullptr : qsum,
                        tp, v.tap_stride, v.tl.off[DFSSM_TAP_GQ], v.tl.off[DFSSM_TAP_S_G],
                        use_mma(c, batch, d.d_inner) ? acc : nullptr, (int)ld_acc, t);
        tm->end(); ++nl;

        tm->begin(DFSSM_KCLASS_PROJ_OUT);
        if (use_mma(c, batch, d.d_inner)) {
            const int rc = launch_proj_mma(c, L.out_sign, L.out_A, d.d_model, d.d_inner, batch, (pdl & 32) != 0);
            if (rc != DFSSM_OK) return rc;
        } else
        DFSSM_LAUNCH_EX(pdl & 32, k_proj, dim3(proj_grid(d.d_model + d.r), (batch + PROJ_BT - 1) / PROJ_BT), PROJ_THREADS, proj_smem(d.d_inner), st,
                        L.out_sign, L.out_A, d.d_model, d.r, d.d_inner, xq, xqp, ldq, qsum, batch, acc, ld_acc, t);
        tm->end(); ++nl;
        if (tp) {
            k_tap_copy_i32<<<dim3((d.d_model + 255) / 256, batch), 256, 0, st>>>(acc, ld_acc, d.d_model, tp,
                                                                                v.tap_stride, v.tl.off[DFSSM_TAP_ACC_OUT]);
            k_tap_copy_i32<<<dim3(1, batch), 64, 0, st>>>(t, T_STRIDE, d.r, tp, v.tap_stride, v.tl.off[DFSSM_TAP_T_OUT]);
            nl += 2;
        }

        tm->begin(DFSSM_KCLASS_EPI_OUT);
        if (fuse) {
            const bool last = l + 1 == d.n_layers;
            launch_epi_norm(L, d, batch, acc, ld_acc, t, sx, u, last ? c->normf_w : c->layers[l + 1].norm_w, xq, ldq, sx,
                            last ? nullptr : acc, last ? nullptr : t, st, (pdl & 64) != 0);
        } else
        launch_epi_out(L, d, batch, acc, ld_acc, t, sx, u, tp, v.tap_stride, v.tl.off[DFSSM_TAP_HIDDEN], st, (pdl & 64) != 0);
        tm->end(); ++nl;
    }

    tm->begin(DFSSM_KCLASS_NORMQUANT);
    if (!fuse)
    DFSSM_LAUNCH_EX(pdl & 1, k_normquant, batch, NQ_THREADS, 0, st, u, d.d_model, c->normf_w, d.d_model, d.eps, xq, mma_in ? nullptr : xqp, ldq, sx,
                    mma_in ? nullptr : qsum,
                    nullptr, 0, 0, 0, nullptr, 0, nullptr);
    tm->end(); ++nl;

    tm->begin(DFSSM_KCLASS_LMHEAD);
    // up to one sequence tile of k_lmhead (8) the warp-per-row dp4a kernel reads the embedding once and beats the tensor-core tiles
    // (cfg 3, us: batch 5 40 / 61, 8 46 / 63, 16 81 / 66)
    if (use_mma(c, batch, d.d_model) && batch > PROJ_BT) {
        DFSSM_LAUNCH_EX(pdl & 2, mma::k_proj_mma<0>, dim3((d.vocab + mma::TM - 1) / mma::TM, (batch + mma::TN - 1) / mma::TN, 1), mma::THREADS, mma::SMEM_BYTES, st,
                        nullptr, c->emb, 0, d.vocab, d.d_model, xq, ldq, batch, nullptr, 0, nullptr, err, logits, sx, c->emb_s);
    } else {
        const int per = LM_THREADS / 32;
        int gx = (d.vocab + per - 1) / per;
        if (gx > 148 * 16) gx = 148 * 16;
        DFSSM_LAUNCH_EX(pdl & 2, k_lmhead, dim3(gx, (batch + PROJ_BT - 1) / PROJ_BT), LM_THREADS, lm_smem(d.d_model), st,
                        c->emb, c->emb_s, d.vocab, d.d_model, xq, ldq, sx, batch, logits);
    }
    tm->end(); ++nl;

    tm->begin(DFSSM_KCLASS_ARGMAX);
    DFSSM_LAUNCH_EX(pdl & 2, k_argmax, batch, AM_THREADS, 0, st, logits, d.vocab, next, tokens, pos, 1);
    tm->end(); ++nl;

    if (fuse) nl -= d.n_layers;                 // the k_normquant launches k_epi_norm4 replaced
    if (n_launch) *n_launch = nl;
    CK(cudaGetLastError());
    return DFSSM_OK;
}

int get_graph(dfssm_ctx* c, int batch, cudaGraphExec_t* out)
{
    dfssm_ctx* ctx = c;
    for (auto& e : c->graphs)
        if (e.batch == batch) { *out = e.exec; return DFSSM_OK; }
    cudaGraph_t graph = nullptr;
    CK(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
    const int rc = enqueue_step(c, batch, nullptr, nullptr);
    cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (rc != DFSSM_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(c, DFSSM_E_CUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(e));
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(c, DFSSM_E_CUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e));
    if (c->graphs.size() >= 16) {               // bounded cache: drop the oldest
        cudaGraphExecDestroy(c->graphs.front().exec);
        c->graphs.erase(c->graphs.begin());
    }
    c->graphs.push_back({ batch, exec });
    *out = exec;
    return DFSSM_OK;
}

}  // namespace


// =================================================================================================
// mega path: one persistent cooperative kernel per batch-1 step
// =================================================================================================
namespace {

// The persistent kernel serves one sequence per launch; a few sequences are stepped by back-to-back launches while that beats the
// kernel chain.  Measured (ms/step, launches of the persistent kernel / chain with tensor-core projections [/ dp4a rows], final
// build): cfg 3 (d_model 2048) batch 2 0.77 / 1.2, 3 1.15 / 1.27, 4 1.53 / 1.29; cfg 4 (2560) batch 2 1.35 / 1.96, 3 2.01 / 2.12,
// 4 2.69 / 2.21; cfg 1 (768) batch 2 0.44 / 0.45 / 0.42, 3 0.66 / 0.47 / 0.46; cfg 0 (256) batch 2 0.057 / 0.046.
int mega_max_batch(const dfssm_ctx* c)
{
    static const int mega_env = getenv("DFSSM_MEGA_MAX") ? atoi(getenv("DFSSM_MEGA_MAX")) : 0;      // measurement switch
    return mega_env > 0 ? mega_env : c->dm.d_model >= 1024 ? 3 : 1;
}
bool use_mega(const dfssm_ctx* c, int batch) { return batch <= mega_max_batch(c) && c->mega_ok && !(c->cfg.flags & DFSSM_FLAG_TAPS && batch > 1); }

int mega_setup(dfssm_ctx* ctx)                      // at create: can this device run the mega grid?
{
    ctx->mega_ok = false;
    if (!ctx->cv.mega_fit) return DFSSM_OK;
    mega::plan(ctx->dm, mega::GRID, ctx->mp);
    int dev = 0, sms = 0, coop = 0, per_sm = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    if (!coop || sms < mega::GRID) return DFSSM_OK;
    ctx->mega_fn = mega::pick_kernel(ctx->dm, (ctx->cfg.flags & DFSSM_FLAG_TAPS) != 0, (ctx->cfg.flags & DFSSM_FLAG_PROF) != 0);
    CK(cudaFuncSetAttribute((const void*)ctx->mega_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->mp.smem_bytes));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)ctx->mega_fn, mega::THREADS, ctx->mp.smem_bytes));
    if (per_sm < 1) return DFSSM_OK;
    ctx->mega_ok = true;
    return DFSSM_OK;
}

// the exchange records of the persistent kernel: everything "not written" (at load, and after a step that was aborted by a
// poll time-out and left half-written records behind)
int mega_init_x(dfssm_ctx* ctx)
{
    const mega::Params& P = ctx->mp;
    const size_t nrec = 2 * (size_t)(P.L > 0 ? P.L : 1);
    mega::k_mega_init_x<<<592, 256, 0, ctx->stream>>>((uint32_t*)(ctx->arena + ctx->cv.m_x), nrec, P.x_main, P.x_small, P.x_A, P.n_early + 1,
                                                      P.x_T, P.n_ttask, (P.n_ttask + 3) / 4 * 4, (P.n_ttask + 3) / 4 * 4 + 4);
    CK(cudaGetLastError());
    return DFSSM_OK;
}

// at load: repack the canonical blob into per-(layer, CTA) chunks and plane-ordered LoRA-down rows
int mega_load(dfssm_ctx* ctx, const std::vector<mega::HostLayer>& HL, const float* normf_w)
{
    if (!ctx->cv.mega_fit) return DFSSM_OK;
    mega::Params& P = ctx->mp;
    const Carve& v = ctx->cv;
    const Dims& d = ctx->dm;
    {
        std::vector<uint8_t> buf((size_t)P.NW * P.chunk_bytes), sbuf((size_t)P.NT * P.schunk_bytes);
        std::vector<int8_t> tmp;
        for (int l = 0; l < d.n_layers; ++l) {
            const float* nn = l + 1 < d.n_layers ? HL[l + 1].norm_w : normf_w;
            for (int c = 0; c < P.NW; ++c) mega::pack_chunk(P, HL[l], nn, c, buf.data() + (size_t)c * P.chunk_bytes);
            for (int s = 0; s < P.NT; ++s) mega::pack_schunk(P, HL[l], s, sbuf.data() + (size_t)s * P.schunk_bytes, tmp);
            CK(cudaMemcpyAsync(ctx->arena + v.m_chunks + (size_t)l * buf.size(), buf.data(), buf.size(), cudaMemcpyHostToDevice, ctx->stream));
            CK(cudaMemcpyAsync(ctx->arena + v.m_schunks + (size_t)l * sbuf.size(), sbuf.data(), sbuf.size(), cudaMemcpyHostToDevice, ctx->stream));
            CK(cudaStreamSynchronize(ctx->stream));
        }
    }
    if (d.n_layers > 0) {      // A_log -> A = -exp(A_log) inside the chunks, with the kernel's own exp
        const size_t n = (size_t)d.n_layers * P.NW * P.nch_max;
        mega::k_mega_prepare<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(ctx->arena + v.m_chunks, (size_t)d.n_layers * P.NW,
                                                                                   P.chunk_bytes, P.c_alog, P.nch_max);
        CK(cudaGetLastError());
    }
    {
        std::vector<uint8_t> buf((size_t)P.blk_bytes);
        for (int l = 0; l < d.n_layers; ++l) {
            mega::pack_block(P, HL[l], buf.data());
            CK(cudaMemcpyAsync(ctx->arena + v.m_blocks + (size_t)l * buf.size(), buf.data(), buf.size(), cudaMemcpyHostToDevice, ctx->stream));
            CK(cudaStreamSynchronize(ctx->stream));
        }
        const int rc = mega_init_x(ctx);        // every exchange word starts as "not written"
        if (rc != DFSSM_OK) return rc;
    }
    // pointers
    const size_t B = ctx->cfg.max_batch;
    P.chunks = ctx->arena + v.m_chunks;
    P.schunks = ctx->arena + v.m_schunks;
    P.ssm = at<float>(ctx, v.ssm);
    P.conv = at<float>(ctx, v.conv);
    P.ssm_lstride = B * v.ssm_elems;
    P.conv_lstride = B * (size_t)d.conv_dim * 4;
    P.emb = ctx->emb; P.emb_s = ctx->emb_s;
    P.first_norm_w = d.n_layers > 0 ? ctx->layers[0].norm_w : ctx->normf_w;
    P.tokens = at<int32_t>(ctx, v.tok);
    P.next = at<int32_t>(ctx, v.next);
    P.tok_out = at<int32_t>(ctx, v.tok);
    P.pos = at<int32_t>(ctx, v.pos);
    P.logits = at<float>(ctx, v.logits);
    P.u_out = at<float>(ctx, v.u);
    P.xbuf = at<uint32_t>(ctx, v.m_x);
    P.blocks = ctx->arena + v.m_blocks;
    P.am_val = at<float>(ctx, v.m_am);
    P.am_idx = (int*)(P.am_val + P.G);
    P.am_count = (unsigned*)(P.am_idx + P.G);
    P.err = at<int>(ctx, v.err);
    const bool taps_on = (ctx->cfg.flags & DFSSM_FLAG_TAPS) != 0;
    P.taps = taps_on ? at<uint8_t>(ctx, v.taps) : nullptr;
    P.tap_lstride = B * (size_t)v.tap_stride;
    P.tl = v.tl;
    P.prof = (ctx->cfg.flags & DFSSM_FLAG_PROF) ? at<unsigned long long>(ctx, v.m_prof) : nullptr;
    return DFSSM_OK;
}

int mega_launch(dfssm_ctx* ctx, int seq = 0)
{
    mega::Params P = ctx->mp;
    if (seq > 0) {                      // this sequence's slices of the per-sequence buffers
        const Dims& d = ctx->dm;
        P.ssm += (size_t)seq * ctx->cv.ssm_elems;
        P.conv += (size_t)seq * d.conv_dim * 4;
        P.tokens += seq; P.next += seq; P.tok_out += seq; P.pos += seq;
        P.logits += (size_t)seq * d.vocab;
        P.u_out += (size_t)seq * d.d_model;
    }
    ctx->epoch += 1;
    P.set = (uint32_t)(ctx->epoch & 1u);       // this step's record set; the kernel resets the other one for the next step
    void* args[] = { &P };
    CK(cudaLaunchCooperativeKernel((const void*)ctx->mega_fn, dim3(P.G), dim3(mega::THREADS), args, P.smem_bytes, ctx->stream));
    return DFSSM_OK;
}

}  // namespace

// =================================================================================================
// prefill: one chunk of T <= CHUNK prompt positions of sequence `seq`, layer by layer (dfssm_prefill.cuh)
// =================================================================================================
namespace {

bool prefill_supported(const Dims& d)
{
    const int nper = d.d_state / prefill::SEQ_LANES;
    return prefill::seq_smem(d) <= 48 * 1024 && d.d_state % prefill::SEQ_LANES == 0 && (nper == 1 || nper == 2 || nper == 4 || nper == 8 || nper == 16) &&
           d.headdim % prefill::SEQ_PB == 0;
}

int prefill_chunk(dfssm_ctx* c, const int32_t* tokens_dev, int T, int seq)
{
    dfssm_ctx* ctx = c;
    static const bool pdl = !(getenv("DFSSM_PDL_MASK") && atoi(getenv("DFSSM_PDL_MASK")) == 0);      // programmatic dependent launch, see enqueue_step
    const Dims& d = c->dm;
    const Carve& v = c->cv;
    cudaStream_t st = c->stream;
    const size_t B = c->cfg.max_batch;
    int32_t* tok = at<int32_t>(c, v.p_tok);
    float* u = at<float>(c, v.p_u);
    int8_t* xq = at<int8_t>(c, v.p_xq);
    int8_t* xqp = at<int8_t>(c, v.p_xqp);
    float* sx = at<float>(c, v.p_sx);
    int32_t* qsum = at<int32_t>(c, v.p_qsum);
    int32_t* acc = at<int32_t>(c, v.p_acc);
    int32_t* t = at<int32_t>(c, v.p_t);
    float* zx = at<float>(c, v.p_zx);
    float* xbc = at<float>(c, v.p_xbc);
    float* dtv = at<float>(c, v.p_dt);
    float* g = at<float>(c, v.p_g);
    int32_t* pos = at<int32_t>(c, v.pos) + seq;
    int* err = at<int>(c, v.err);
    const int ldq = (int)v.ldq, ld_acc = (int)v.ld_acc;
    auto proj = [&](const uint32_t* sign, const int8_t* A, int rows, int K) {
        if (use_mma(c, T, K)) {
            const int mt = (rows + d.r + mma::TM - 1) / mma::TM, nt = (T + mma::TN - 1) / mma::TN, nchunk = (K + mma::KC - 1) / mma::KC;
            int ks = (148 * MMA_CTAS_PER_SM) / (mt * nt);
            if (ks < 1) ks = 1;
            if (ks > nchunk) ks = nchunk;
            DFSSM_MMA_LAUNCH(pdl, d.fmt, dim3(mt, nt, ks), st, sign, A, rows, d.r, K, xq, ldq, T, acc, ld_acc, t, err, nullptr, nullptr, nullptr);
        } else {
            DFSSM_LAUNCH_EX(pdl, k_proj, dim3(proj_grid(rows + d.r), (T + PROJ_BT - 1) / PROJ_BT), PROJ_THREADS, proj_smem(K), st, sign, A, rows, d.r, K, xq, xqp, ldq, qsum,
                                                                                                              T, acc, ld_acc, t);
        }
    };
    CK(cudaMemcpyAsync(tok, tokens_dev, sizeof(int32_t) * (size_t)T, cudaMemcpyDeviceToDevice, st));
    k_embed<<<dim3((d.d_model + 255) / 256, T), 256, 0, st>>>(tok, c->emb, c->emb_s, d.vocab, d.d_model, u, err);
    for (int l = 0; l < d.n_layers; ++l) {
        const LayerW& L = c->layers[l];
        uint8_t* ssm_b = c->arena + v.ssm + ((size_t)l * B + seq) * v.ssm_elems * v.ssm_esize;
        float* ring = at<float>(c, v.conv) + ((size_t)l * B + seq) * (size_t)d.conv_dim * 4;
        DFSSM_LAUNCH_EX(pdl, k_normquant, T, NQ_THREADS, 0, st, u, d.d_model, L.norm_w, d.d_model, d.eps, xq, xqp, ldq, sx, qsum, nullptr, 0, 0, 0,
                                              use_mma(c, T, d.d_model) ? acc : nullptr, ld_acc, t);
        proj(L.in_sign, L.in_A, d.d_in_proj, d.d_model);
        {
            const dim3 g4((d.d_in_proj + FIN_THREADS - 1) / FIN_THREADS, T);
            switch (d.r) {
                case 8:
                    if (d.fmt & 2) DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_epi4<2, true>), g4, FIN_THREADS, 0, st, L, d, acc, ld_acc, t, sx, zx, ld_acc);
                    else DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_epi4<2, false>), g4, FIN_THREADS, 0, st, L, d, acc, ld_acc, t, sx, zx, ld_acc);
                    break;
                case 16:
                    if (d.fmt & 2) DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_epi4<4, true>), g4, FIN_THREADS, 0, st, L, d, acc, ld_acc, t, sx, zx, ld_acc);
                    else DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_epi4<4, false>), g4, FIN_THREADS, 0, st, L, d, acc, ld_acc, t, sx, zx, ld_acc);
                    break;
                case 32:
                    if (d.fmt & 2) DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_epi4<8, true>), g4, FIN_THREADS, 0, st, L, d, acc, ld_acc, t, sx, zx, ld_acc);
                    else DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_epi4<8, false>), g4, FIN_THREADS, 0, st, L, d, acc, ld_acc, t, sx, zx, ld_acc);
                    break;
                case 64:
                    if (d.fmt & 2) DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_epi4<16, true>), g4, FIN_THREADS, 0, st, L, d, acc, ld_acc, t, sx, zx, ld_acc);
                    else DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_epi4<16, false>), g4, FIN_THREADS, 0, st, L, d, acc, ld_acc, t, sx, zx, ld_acc);
                    break;
                default:
                    prefill::k_pf_epi<<<dim3((d.d_in_proj + prefill::EPI_T - 1) / prefill::EPI_T, T), prefill::EPI_T, 0, st>>>(L, d, acc, ld_acc, t, sx, zx,
                                                                                                                        ld_acc);
            }
        }
        DFSSM_LAUNCH_EX(pdl, prefill::k_pf_conv, dim3((d.conv_dim + d.nheads + prefill::CONV_T - 1) / prefill::CONV_T, T), prefill::CONV_T, 0, st, L, d, zx, ld_acc, T, ring, pos, xbc,
                                                                                                                               dtv);
        DFSSM_LAUNCH_EX(pdl, prefill::k_pf_ring, (d.conv_dim + 255) / 256, 256, 0, st, d, zx, ld_acc, T, ring, pos);
        {
            const dim3 gr(d.nheads * (d.headdim / prefill::SEQ_PB));
            const size_t sm = prefill::seq_smem(d);
#define DFSSM_PF_SSM(N_)                                                                                                             \
    if (v.ssm_esize == 2) DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_ssm<N_, __half>), gr, prefill::SEQ_T, sm, st, L, d, zx, ld_acc, xbc, dtv, T, (__half*)ssm_b, g); \
    else DFSSM_LAUNCH_EX(pdl, (prefill::k_pf_ssm<N_, float>), gr, prefill::SEQ_T, sm, st, L, d, zx, ld_acc, xbc, dtv, T, (float*)ssm_b, g)
            switch (d.d_state / prefill::SEQ_LANES) {
                case 1: DFSSM_PF_SSM(1); break;
                case 2: DFSSM_PF_SSM(2); break;
                case 4: DFSSM_PF_SSM(4); break;
                case 8: DFSSM_PF_SSM(8); break;
                default: DFSSM_PF_SSM(16); break;
            }
#undef DFSSM_PF_SSM
        }
        DFSSM_LAUNCH_EX(pdl, k_normquant, T, NQ_THREADS, 0, st, g, d.d_inner, L.gnorm_w, d.d_inner, d.eps, xq, xqp, ldq, sx, qsum, nullptr, 0, 0, 0,
                                              use_mma(c, T, d.d_inner) ? acc : nullptr, ld_acc, t);
        proj(L.out_sign, L.out_A, d.d_model, d.d_inner);
        launch_epi_out(L, d, T, acc, ld_acc, t, sx, u, nullptr, 0, 0, st, pdl);
    }
    // the last position: hidden state, logits and greedy token of the sequence; the conv ring position advances by T
    const float* u_last = u + (size_t)(T - 1) * d.d_model;
    float* logits = at<float>(c, v.logits) + (size_t)seq * d.vocab;
    prefill::k_pf_copy_hidden<<<(d.d_model + 255) / 256, 256, 0, st>>>(u_last, at<float>(c, v.u) + (size_t)seq * d.d_model, d.d_model);
    k_normquant<<<1, NQ_THREADS, 0, st>>>(u_last, d.d_model, c->normf_w, d.d_model, d.eps, xq, xqp, ldq, sx, qsum, nullptr, 0, 0, 0);
    {
        const int per = LM_THREADS / 32;
        int gx = (d.vocab + per - 1) / per;
        if (gx > 148 * 16) gx = 148 * 16;
        k_lmhead<<<dim3(gx, 1), LM_THREADS, lm_smem(d.d_model), st>>>(c->emb, c->emb_s, d.vocab, d.d_model, xq, ldq, sx, 1, logits);
    }
    k_argmax<<<1, AM_THREADS, 0, st>>>(logits, d.vocab, at<int32_t>(c, v.next) + seq, at<int32_t>(c, v.tok) + seq, pos, T);
    CK(cudaGetLastError());
    return DFSSM_OK;
}

}  // namespace

// =================================================================================================
// exported C ABI
// =================================================================================================
extern "C" {

size_t dfssm_arena_bytes(const dfssm_config* cfg)
{
    if (!valid_cfg(cfg)) return 0;
    return carve(*cfg).total;
}

int dfssm_create(const dfssm_config* cfg, void* dev_arena, size_t arena_bytes, void* cuda_stream, dfssm_ctx** out)
{
    if (!out) return DFSSM_E_ARG;
    *out = nullptr;
    if (!valid_cfg(cfg) || !dev_arena || ((uintptr_t)dev_arena % ARENA_ALIGN)) return DFSSM_E_ARG;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return DFSSM_E_CUDA;
    if (prop.major != 10) return DFSSM_E_ARCH;
    dfssm_ctx* ctx = new (std::nothrow) dfssm_ctx();
    if (!ctx) return DFSSM_E_ARG;
    ctx->cfg = *cfg;
    ctx->dm = make_dims(*cfg);
    ctx->cv = carve(*cfg);
    ctx->arena = (uint8_t*)dev_arena;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->loaded = false;
    ctx->failed = false;
    ctx->last_batch = 0;
    ctx->pinned_tok = nullptr;
    ctx->pinned_err = nullptr;
    ctx->err[0] = 0;
    ctx->mega_ok = false;
    ctx->epoch = 0;
    *out = ctx;                       // handed out even on failure below so last_error can be read
    if (arena_bytes < ctx->cv.total)
        return fail(ctx, DFSSM_E_SIZE, "arena too small: %zu < %zu", arena_bytes, ctx->cv.total);
    CK(cudaMallocHost((void**)&ctx->pinned_tok, sizeof(int32_t) * 2 * (size_t)cfg->max_batch));
    CK(cudaMallocHost((void**)&ctx->pinned_err, sizeof(int)));
    CK(cudaFuncSetAttribute(k_proj, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)proj_smem(8192)));
    CK(cudaFuncSetAttribute(k_lmhead, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lm_smem(8192)));
    CK(cudaFuncSetAttribute(mma::k_proj_mma<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mma::SMEM_BYTES));
    CK(cudaFuncSetAttribute(mma::k_proj_mma<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mma::SMEM_BYTES));
    CK(cudaFuncSetAttribute(mma::k_proj_mma<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mma::SMEM_BYTES));
    CK(cudaFuncSetAttribute(mma::k_proj_mma<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mma::SMEM_BYTES));
    {
        const int rc = mega_setup(ctx);
        if (rc != DFSSM_OK) return rc;
    }
    // zero everything behind the weights: state, ring positions, activations, error flag
    CK(cudaMemsetAsync(ctx->arena + ctx->cv.ssm, 0, ctx->cv.total - ctx->cv.ssm, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return DFSSM_OK;
}

int dfssm_load_weights(dfssm_ctx* ctx, const void* host_blob, size_t nbytes)
{
    if (!ctx || !host_blob) return DFSSM_E_ARG;
    const Dims& d = ctx->dm;
    const uint8_t* hb = (const uint8_t*)host_blob;
    if (nbytes < 256 || memcmp(hb, "DFSSMW1\0", 8) != 0) return fail(ctx, DFSSM_E_SIZE, "bad magic or short blob");
    uint32_t ver, hfmt; int32_t hdr[9]; float eps; uint64_t total;
    memcpy(&hfmt, hb + 52, 4);
    memcpy(&ver, hb + 8, 4); memcpy(hdr, hb + 12, 36); memcpy(&eps, hb + 48, 4); memcpy(&total, hb + 56, 8);
    if (ver != 1) return fail(ctx, DFSSM_E_ARG, "unsupported blob version %u", ver);
    const int32_t want[9] = { d.n_layers, d.d_model, d.d_inner, d.headdim, d.d_state, d.ngroups, 4, d.vocab, d.r };
    for (int i = 0; i < 9; ++i)
        if (hdr[i] != want[i]) return fail(ctx, DFSSM_E_ARG, "blob header field %d = %d does not match the config (%d)", i, hdr[i], want[i]);
    if (eps != d.eps) return fail(ctx, DFSSM_E_ARG, "blob norm_eps does not match the config");
    if ((int)hfmt != d.fmt)
        return fail(ctx, DFSSM_E_ARG, "blob weight format %u (bit 0: 17-level scaffold, bit 1: int4 LoRA) does not match the config flags (%d)", hfmt, d.fmt);
    const size_t expect = blob_bytes_for(d);
    if (total != nbytes || nbytes != expect)
        return fail(ctx, DFSSM_E_SIZE, "blob size %zu does not match its header (%llu) / the shape (%zu)", nbytes,
                    (unsigned long long)total, expect);

    uint8_t* db = ctx->arena + ctx->cv.blob;
    CK(cudaMemcpyAsync(db, hb, nbytes, cudaMemcpyHostToDevice, ctx->stream));
    BlobWalk w;
    const size_t dm = d.d_model, di = d.d_inner, dip = d.d_in_proj, r = d.r, cd = d.conv_dim, nh = d.nheads;
    const size_t pl = (d.fmt & 1) ? 5 : 1, ld = (d.fmt & 2) ? 2 : 1;
    ctx->layers.assign((size_t)d.n_layers, LayerW());
    std::vector<mega::HostLayer> HL((size_t)d.n_layers);
    for (int l = 0; l < d.n_layers; ++l) {
        LayerW& L = ctx->layers[l];
        L.norm_w = (const float*)(db + w.take(4 * dm));
        L.in_sign = (const uint32_t*)(db + w.take(4 * dip * (dm / 32) * pl));
        L.in_row_scale = (const __half*)(db + w.take(2 * dip));
        L.in_A = (const int8_t*)(db + w.take(r * dm / ld));
        L.in_a_s = (const float*)(db + w.take(4 * r));
        L.in_B = (const int8_t*)(db + w.take(dip * r / ld));
        L.in_b_s = (const float*)(db + w.take(4 * dip));
        L.conv_w = (const float*)(db + w.take(16 * cd));
        L.conv_b = (const float*)(db + w.take(4 * cd));
        L.A_log = (const float*)(db + w.take(4 * nh));
        L.dt_bias = (const float*)(db + w.take(4 * nh));
        L.D = (const float*)(db + w.take(4 * nh));
        L.gnorm_w = (const float*)(db + w.take(4 * di));
        L.out_sign = (const uint32_t*)(db + w.take(4 * dm * (di / 32) * pl));
        L.out_row_scale = (const __half*)(db + w.take(2 * dm));
        L.out_A = (const int8_t*)(db + w.take(r * di / ld));
        L.out_a_s = (const float*)(db + w.take(4 * r));
        L.out_B = (const int8_t*)(db + w.take(dm * r / ld));
        L.out_b_s = (const float*)(db + w.take(4 * dm));
        // the same tensors in the host blob (for the mega repack)
        mega::HostLayer& H = HL[l];
        auto hp = [&](const void* dev_ptr) { return hb + ((const uint8_t*)dev_ptr - db); };
        H.norm_w = (const float*)hp(L.norm_w);
        H.in_sign = (const uint32_t*)hp(L.in_sign); H.in_row_scale = (const uint16_t*)hp(L.in_row_scale);
        H.in_A = (const int8_t*)hp(L.in_A); H.in_a_s = (const float*)hp(L.in_a_s);
        H.in_B = (const int8_t*)hp(L.in_B); H.in_b_s = (const float*)hp(L.in_b_s);
        H.conv_w = (const float*)hp(L.conv_w); H.conv_b = (const float*)hp(L.conv_b);
        H.A_log = (const float*)hp(L.A_log); H.dt_bias = (const float*)hp(L.dt_bias); H.D = (const float*)hp(L.D);
        H.gnorm_w = (const float*)hp(L.gnorm_w);
        H.out_sign = (const uint32_t*)hp(L.out_sign); H.out_row_scale = (const uint16_t*)hp(L.out_row_scale);
        H.out_A = (const int8_t*)hp(L.out_A); H.out_a_s = (const float*)hp(L.out_a_s);
        H.out_B = (const int8_t*)hp(L.out_B); H.out_b_s = (const float*)hp(L.out_b_s);
    }
    ctx->emb = (const int8_t*)(db + w.take((size_t)d.vocab * dm));
    ctx->emb_s = (const float*)(db + w.take(4 * (size_t)d.vocab));
    ctx->normf_w = (const float*)(db + w.take(4 * dm));
    CK(cudaStreamSynchronize(ctx->stream));
    {
        const int rc = mega_load(ctx, HL, (const float*)(hb + ((const uint8_t*)ctx->normf_w - db)));
        if (rc != DFSSM_OK) return rc;
    }
    for (auto& e : ctx->graphs) cudaGraphExecDestroy(e.exec);
    ctx->graphs.clear();
    ctx->blob_bytes = nbytes;
    ctx->loaded = true;
    return DFSSM_OK;
}

int dfssm_reset_state(dfssm_ctx* ctx, int seq)
{
    if (!ctx) return DFSSM_E_ARG;
    if (seq >= ctx->cfg.max_batch) return fail(ctx, DFSSM_E_ARG, "seq_index out of range");
    const Dims& d = ctx->dm;
    const Carve& v = ctx->cv;
    const size_t B = ctx->cfg.max_batch, nl = d.n_layers > 0 ? d.n_layers : 1;
    if (seq < 0) {
        CK(cudaMemsetAsync(ctx->arena + v.ssm, 0, nl * B * v.ssm_elems * v.ssm_esize, ctx->stream));
        CK(cudaMemsetAsync(ctx->arena + v.conv, 0, nl * B * (size_t)d.conv_dim * 16, ctx->stream));
        // the exchange records of the persistent kernel go back to "nothing written" too (matters only after a step that
        // was aborted by a poll time-out and left half-written records behind)
        if (v.mega_fit && ctx->loaded) {
            const int rc = mega_init_x(ctx);
            if (rc != DFSSM_OK) return rc;
        }
        ctx->failed = false;
        return DFSSM_OK;
    }
    // one sequence of every layer: strided 2-D memsets (rows = layers)
    CK(cudaMemset2DAsync(ctx->arena + v.ssm + (size_t)seq * v.ssm_elems * v.ssm_esize, B * v.ssm_elems * v.ssm_esize, 0,
                         v.ssm_elems * v.ssm_esize, nl, ctx->stream));
    CK(cudaMemset2DAsync(ctx->arena + v.conv + (size_t)seq * d.conv_dim * 16, B * (size_t)d.conv_dim * 16, 0,
                         (size_t)d.conv_dim * 16, nl, ctx->stream));
    return DFSSM_OK;
}

int dfssm_step(dfssm_ctx* ctx, const int32_t* tokens_dev, int batch)
{
    if (!ctx || !tokens_dev) return DFSSM_E_ARG;
    if (!ctx->loaded) return fail(ctx, DFSSM_E_STATE, "dfssm_step before dfssm_load_weights");
    if (batch < 1 || batch > ctx->cfg.max_batch) return fail(ctx, DFSSM_E_ARG, "batch %d outside [1, %d]", batch, ctx->cfg.max_batch);
    if (ctx->failed) return fail(ctx, DFSSM_E_STATE, "an earlier step timed out on the device: call dfssm_reset_state(ctx, -1) first");
    // the step reads its tokens from the arena's token buffer.  After a step that buffer already
    // holds the greedy tokens, so feeding dfssm_next_tokens' pointer back costs no copy at all.
    int32_t* tok = at<int32_t>(ctx, ctx->cv.tok);
    const int32_t* next = at<int32_t>(ctx, ctx->cv.next);
    const bool resident = tokens_dev == tok || (tokens_dev == next && batch <= ctx->last_batch);
    if (!resident)
        CK(cudaMemcpyAsync(tok, tokens_dev, sizeof(int32_t) * (size_t)batch, cudaMemcpyDeviceToDevice, ctx->stream));
    ctx->last_batch = batch;
    if (use_mega(ctx, batch)) {
        for (int seq = 0; seq < batch; ++seq) {
            const int rc = mega_launch(ctx, seq);
            if (rc != DFSSM_OK) return rc;
        }
        return DFSSM_OK;
    }
    if (ctx->cfg.flags & (DFSSM_FLAG_NO_GRAPH | DFSSM_FLAG_TAPS)) return enqueue_step(ctx, batch, nullptr, nullptr);
    cudaGraphExec_t exec;
    const int rc = get_graph(ctx, batch, &exec);
    if (rc != DFSSM_OK) return rc;
    CK(cudaGraphLaunch(exec, ctx->stream));
    return DFSSM_OK;
}

int dfssm_prefill(dfssm_ctx* ctx, const int32_t* tokens_dev, int n_tokens, int seq)
{
    if (!ctx || !tokens_dev) return DFSSM_E_ARG;
    if (!ctx->loaded) return fail(ctx, DFSSM_E_STATE, "dfssm_prefill before dfssm_load_weights");
    if (n_tokens < 1 || seq < 0 || seq >= ctx->cfg.max_batch) return fail(ctx, DFSSM_E_ARG, "n_tokens %d / seq %d out of range", n_tokens, seq);
    if (ctx->failed) return fail(ctx, DFSSM_E_STATE, "an earlier step timed out on the device: call dfssm_reset_state(ctx, -1) first");
    if (ctx->last_batch < seq + 1) ctx->last_batch = seq + 1;
    if (!prefill_supported(ctx->dm) || (ctx->cfg.flags & DFSSM_FLAG_TAPS)) {
        // shapes the serial-in-t state kernel does not cover (d_state not a multiple of 16), or taps wanted: token by token
        // through the persistent kernel / chain of the step path (same results by construction)
        if (seq != 0 || ctx->cfg.max_batch != 1) return fail(ctx, DFSSM_E_ARG, "this shape prefills only through dfssm_step");
        for (int i = 0; i < n_tokens; ++i) {
            const int rc = dfssm_step(ctx, tokens_dev + i, 1);
            if (rc != DFSSM_OK) return rc;
        }
        return DFSSM_OK;
    }
    for (int i = 0; i < n_tokens; i += prefill::CHUNK) {
        const int T = n_tokens - i < prefill::CHUNK ? n_tokens - i : prefill::CHUNK;
        const int rc = prefill_chunk(ctx, tokens_dev + i, T, seq);
        if (rc != DFSSM_OK) return rc;
    }
    return DFSSM_OK;
}

int dfssm_sample(dfssm_ctx* ctx, int batch, float temperature, int top_k, const float* uniform_dev)
{
    if (!ctx || !uniform_dev) return DFSSM_E_ARG;
    if (!ctx->loaded) return fail(ctx, DFSSM_E_STATE, "dfssm_sample before dfssm_load_weights");
    if (batch < 1 || batch > ctx->cfg.max_batch) return fail(ctx, DFSSM_E_ARG, "batch %d outside [1, %d]", batch, ctx->cfg.max_batch);
    if (top_k < 1 || top_k > SAMPLE_KMAX) return fail(ctx, DFSSM_E_ARG, "top_k %d outside [1, %d]", top_k, SAMPLE_KMAX);
    k_sample<<<batch, SAMPLE_THREADS, 0, ctx->stream>>>(at<float>(ctx, ctx->cv.logits), ctx->dm.vocab, temperature, top_k, uniform_dev,
                                                        at<int32_t>(ctx, ctx->cv.next), at<int32_t>(ctx, ctx->cv.tok));
    CK(cudaGetLastError());
    return DFSSM_OK;
}

int dfssm_step_host(dfssm_ctx* ctx, const int32_t* tokens_host, int batch, int32_t* next_host, float* logits_host)
{
    if (!ctx || !tokens_host || !next_host) return DFSSM_E_ARG;
    if (batch < 1 || batch > ctx->cfg.max_batch) return fail(ctx, DFSSM_E_ARG, "batch %d outside [1, %d]", batch, ctx->cfg.max_batch);
    int32_t* tok_dev = at<int32_t>(ctx, ctx->cv.tok);
    memcpy(ctx->pinned_tok, tokens_host, sizeof(int32_t) * (size_t)batch);
    CK(cudaMemcpyAsync(tok_dev, ctx->pinned_tok, sizeof(int32_t) * (size_t)batch, cudaMemcpyHostToDevice, ctx->stream));
    const int rc = dfssm_step(ctx, tok_dev, batch);
    if (rc != DFSSM_OK) return rc;
    int32_t* stage = ctx->pinned_tok + ctx->cfg.max_batch;
    CK(cudaMemcpyAsync(stage, at<int32_t>(ctx, ctx->cv.next), sizeof(int32_t) * (size_t)batch, cudaMemcpyDeviceToHost, ctx->stream));
    if (logits_host)
        CK(cudaMemcpyAsync(logits_host, at<float>(ctx, ctx->cv.logits), sizeof(float) * (size_t)batch * ctx->dm.vocab,
                           cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    memcpy(next_host, stage, sizeof(int32_t) * (size_t)batch);
    return DFSSM_OK;
}

int dfssm_logits(dfssm_ctx* ctx, const float** p)
{
    if (!ctx || !p) return DFSSM_E_ARG;
    *p = at<float>(ctx, ctx->cv.logits);
    return DFSSM_OK;
}

int dfssm_next_tokens(dfssm_ctx* ctx, const int32_t** p)
{
    if (!ctx || !p) return DFSSM_E_ARG;
    *p = at<int32_t>(ctx, ctx->cv.next);
    return DFSSM_OK;
}

int dfssm_hidden(dfssm_ctx* ctx, const float** p)
{
    if (!ctx || !p) return DFSSM_E_ARG;
    *p = at<float>(ctx, ctx->cv.u);
    return DFSSM_OK;
}

int dfssm_debug_tensor(dfssm_ctx* ctx, int layer, int which, int seq, const void** dev, size_t* nbytes)
{
    if (!ctx || !dev) return DFSSM_E_ARG;
    if (!(ctx->cfg.flags & DFSSM_FLAG_TAPS)) return fail(ctx, DFSSM_E_STATE, "context created without DFSSM_FLAG_TAPS");
    if (layer < 0 || layer >= ctx->dm.n_layers || which < 0 || which >= DFSSM_TAP_COUNT || seq < 0 || seq >= ctx->cfg.max_batch)
        return fail(ctx, DFSSM_E_ARG, "tap index out of range");
    const Carve& v = ctx->cv;
    *dev = ctx->arena + v.taps + ((size_t)layer * ctx->cfg.max_batch + seq) * v.tap_stride + v.tl.off[which];
    if (nbytes) *nbytes = tap_bytes(ctx->dm, which);
    return DFSSM_OK;
}

static int state_copy(dfssm_ctx* ctx, int layer, int seq, float* ssm_h, size_t ssm_bytes, float* conv_h,
                      size_t conv_bytes, bool to_host)
{
    if (!ctx) return DFSSM_E_ARG;
    const Dims& d = ctx->dm;
    const Carve& v = ctx->cv;
    if (layer < 0 || layer >= d.n_layers || seq < 0 || seq >= ctx->cfg.max_batch) return fail(ctx, DFSSM_E_ARG, "state index out of range");
    const size_t B = ctx->cfg.max_batch;
    if (ssm_h && ssm_bytes != v.ssm_elems * 4) return fail(ctx, DFSSM_E_SIZE, "ssm state is %zu bytes", v.ssm_elems * 4);
    if (conv_h && conv_bytes != (size_t)d.conv_dim * 12) return fail(ctx, DFSSM_E_SIZE, "conv state is %zu bytes", (size_t)d.conv_dim * 12);
    CK(cudaStreamSynchronize(ctx->stream));
    uint8_t* ssm_d = ctx->arena + v.ssm + ((size_t)layer * B + seq) * v.ssm_elems * v.ssm_esize;
    float* ring_d = at<float>(ctx, v.conv) + ((size_t)layer * B + seq) * (size_t)d.conv_dim * 4;
    if (ssm_h) {
        if (v.ssm_esize == 4) {
            if (to_host) CK(cudaMemcpy(ssm_h, ssm_d, ssm_bytes, cudaMemcpyDeviceToHost));
            else CK(cudaMemcpy(ssm_d, ssm_h, ssm_bytes, cudaMemcpyHostToDevice));
        } else {                               // fp16 state format: the host view stays fp32 (set: rounded to nearest even)
            std::vector<__half> tmp(v.ssm_elems);
            if (to_host) {
                CK(cudaMemcpy(tmp.data(), ssm_d, v.ssm_elems * 2, cudaMemcpyDeviceToHost));
                for (size_t i = 0; i < v.ssm_elems; ++i) ssm_h[i] = __half2float(tmp[i]);
            } else {
                for (size_t i = 0; i < v.ssm_elems; ++i) tmp[i] = __float2half_rn(ssm_h[i]);
                CK(cudaMemcpy(ssm_d, tmp.data(), v.ssm_elems * 2, cudaMemcpyHostToDevice));
            }
        }
    }
    if (conv_h) {
        // ring <-> canonical [conv_dim][3] oldest first: the next step writes slot pos, so the three
        // live samples are slots pos+1, pos+2, pos+3 (mod 4), oldest first
        int32_t pos = 0;
        CK(cudaMemcpy(&pos, at<int32_t>(ctx, v.pos) + seq, 4, cudaMemcpyDeviceToHost));
        pos &= 3;
        std::vector<float> ring((size_t)d.conv_dim * 4);
        if (to_host) {
            CK(cudaMemcpy(ring.data(), ring_d, ring.size() * 4, cudaMemcpyDeviceToHost));
            for (int c = 0; c < d.conv_dim; ++c)
                for (int j = 0; j < 3; ++j) conv_h[3 * (size_t)c + j] = ring[4 * (size_t)c + ((pos + 1 + j) & 3)];
        } else {
            for (int c = 0; c < d.conv_dim; ++c) {
                ring[4 * (size_t)c + pos] = 0.0f;
                for (int j = 0; j < 3; ++j) ring[4 * (size_t)c + ((pos + 1 + j) & 3)] = conv_h[3 * (size_t)c + j];
            }
            CK(cudaMemcpy(ring_d, ring.data(), ring.size() * 4, cudaMemcpyHostToDevice));
        }
    }
    return DFSSM_OK;
}

int dfssm_get_state(dfssm_ctx* ctx, int layer, int seq, float* ssm_host, size_t ssm_bytes, float* conv_host, size_t conv_bytes)
{
    return state_copy(ctx, layer, seq, ssm_host, ssm_bytes, conv_host, conv_bytes, true);
}

int dfssm_set_state(dfssm_ctx* ctx, int layer, int seq, const float* ssm_host, size_t ssm_bytes, const float* conv_host, size_t conv_bytes)
{
    return state_copy(ctx, layer, seq, const_cast<float*>(ssm_host), ssm_bytes, const_cast<float*>(conv_host), conv_bytes, false);
}

int dfssm_debug_profile(dfssm_ctx* ctx, uint64_t* stamps_host, size_t nbytes, int32_t* dims)
{
    if (!ctx || !dims) return DFSSM_E_ARG;
    if (!(ctx->cfg.flags & DFSSM_FLAG_PROF) || !ctx->mega_ok || !ctx->loaded)
        return fail(ctx, DFSSM_E_STATE, "no profile: context created without DFSSM_FLAG_PROF, or the persistent kernel is not in use");
    dims[0] = ctx->mp.G; dims[1] = ctx->mp.L + 1; dims[2] = mega::PROF_NPH;
    const size_t need = (size_t)dims[0] * dims[1] * dims[2] * 8;
    if (!stamps_host) return DFSSM_OK;
    if (nbytes != need) return fail(ctx, DFSSM_E_SIZE, "profile is %zu bytes", need);
    CK(cudaStreamSynchronize(ctx->stream));
    CK(cudaMemcpy(stamps_host, ctx->arena + ctx->cv.m_prof, need, cudaMemcpyDeviceToHost));
    return DFSSM_OK;
}

int dfssm_sync(dfssm_ctx* ctx)
{
    if (!ctx) return DFSSM_E_ARG;
    int* err_d = at<int>(ctx, ctx->cv.err);
    CK(cudaMemcpyAsync(ctx->pinned_err, err_d, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (*ctx->pinned_err) {
        const int bits = *ctx->pinned_err;
        CK(cudaMemsetAsync(err_d, 0, sizeof(int), ctx->stream));
        if (bits & 6) ctx->failed = true;      // sticky: dfssm_step refuses until dfssm_reset_state(ctx, -1)
        if (bits & 2) return fail(ctx, DFSSM_E_CUDA, "the persistent step kernel timed out waiting for an exchange between CTAs");
        if (bits & 4) return fail(ctx, DFSSM_E_CUDA, "a tensor-core projection timed out waiting for its MMAs");
        return fail(ctx, DFSSM_E_TOKEN, "a token id outside [0, vocab) was clamped");
    }
    return DFSSM_OK;
}

int dfssm_launches_per_step(dfssm_ctx* ctx, int batch)
{
    if (!ctx || batch < 1) return DFSSM_E_ARG;
    if (use_mega(ctx, batch)) return batch;
    const int per_layer = (ctx->cfg.flags & DFSSM_FLAG_TAPS) ? 11 : 7;
    return 1 + ctx->dm.n_layers * per_layer + 3 - (fused_epi_norm(ctx, batch) ? ctx->dm.n_layers : 0);
}

int dfssm_time_kernels(dfssm_ctx* ctx, const int32_t* tokens_dev, int batch, int iters, float* out_us)
{
    if (!ctx || !tokens_dev || !out_us || iters < 1) return DFSSM_E_ARG;
    if (!ctx->loaded) return fail(ctx, DFSSM_E_STATE, "dfssm_time_kernels before dfssm_load_weights");
    if (batch < 1 || batch > ctx->cfg.max_batch) return fail(ctx, DFSSM_E_ARG, "batch out of range");
    double sum[DFSSM_KCLASS_COUNT] = { 0 };
    if (use_mega(ctx, batch)) {                  // one kernel: time it with events on the library's stream
        cudaEvent_t a, b;
        CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
        CK(cudaMemcpyAsync(at<int32_t>(ctx, ctx->cv.tok), tokens_dev, sizeof(int32_t) * (size_t)batch, cudaMemcpyDeviceToDevice, ctx->stream));
        for (int k = 0; k < DFSSM_KCLASS_COUNT; ++k) out_us[k] = 0.0f;
        for (int it = 0; it < iters; ++it) {
            CK(cudaEventRecord(a, ctx->stream));
            for (int seq = 0; seq < batch; ++seq) {
                const int rc = mega_launch(ctx, seq);
                if (rc != DFSSM_OK) return rc;
            }
            CK(cudaEventRecord(b, ctx->stream));
            CK(cudaEventSynchronize(b));
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, a, b));
            sum[DFSSM_KCLASS_MEGA] += 1e3 * ms;
        }
        cudaEventDestroy(a); cudaEventDestroy(b);
        out_us[DFSSM_KCLASS_MEGA] = (float)(sum[DFSSM_KCLASS_MEGA] / iters);
        return DFSSM_OK;
    }
    for (int it = 0; it < iters; ++it) {
        KTimer tm;
        tm.on = true;
        tm.st = ctx->stream;
        CK(cudaMemcpyAsync(at<int32_t>(ctx, ctx->cv.tok), tokens_dev, sizeof(int32_t) * (size_t)batch,
                           cudaMemcpyDeviceToDevice, ctx->stream));
        const int rc = enqueue_step(ctx, batch, &tm, nullptr);
        cudaError_t e = cudaStreamSynchronize(ctx->stream);
        if (rc == DFSSM_OK && e == cudaSuccess)
            for (size_t i = 0; i < tm.cls.size(); ++i) {
                float ms = 0.f;
                cudaEventElapsedTime(&ms, tm.ev[2 * i], tm.ev[2 * i + 1]);
                sum[tm.cls[i]] += 1e3 * ms;
            }
        for (auto ev : tm.ev) cudaEventDestroy(ev);
        if (rc != DFSSM_OK) return rc;
        if (e != cudaSuccess) return fail(ctx, DFSSM_E_CUDA, "sync failed: %s", cudaGetErrorString(e));
    }
    for (int k = 0; k < DFSSM_KCLASS_COUNT; ++k) out_us[k] = (float)(sum[k] / iters);
    return DFSSM_OK;
}

const char* dfssm_last_error(const dfssm_ctx* ctx) { return ctx ? ctx->err : ""; }

void dfssm_destroy(dfssm_ctx* ctx)
{
    if (!ctx) return;
    for (auto& e : ctx->graphs) cudaGraphExecDestroy(e.exec);
    if (ctx->pinned_tok) cudaFreeHost(ctx->pinned_tok);
    if (ctx->pinned_err) cudaFreeHost(ctx->pinned_err);
    delete ctx;
}

}  // extern "C"
