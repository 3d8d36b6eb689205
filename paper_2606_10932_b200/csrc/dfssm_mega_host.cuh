// Host side of the mega path: the per-(layer, CTA) chunk layout, the shared-memory plan, and the
// load-time repack of the canonical blob (DESIGN.md sections 3 and 6) into that layout.
#pragma once
#include <cstdlib>
#include <cstring>
#include <vector>

#include "dfssm_mega.cuh"

namespace dfssm {
namespace mega {

constexpr size_t SMEM_LIMIT = 232448 - 1024;    // 227 KB opt-in maximum minus the kernel's static shared memory

inline uint32_t up32(uint32_t x, uint32_t a) { return (x + a - 1) / a * a; }

// workers of a shape: 128 whenever that deals whole groups of 4 to every worker (all BASELINE shapes), else the count in
// [112, 128] with the least sign-row work on the busiest worker
inline int pick_workers(const Dims& d)
{
    if ((d.d_inner / 4) % NW_CT == 0 || d.d_inner / 4 < NW_CT) return NW_CT;
    int best = NW_CT;
    long long best_cost = -1;
    for (int nw = 128; nw >= 112; nw -= 4) {         // <= 128: a warp polls the workers' maxima with one 16-byte chunk per lane
        const long long cost = (long long)own_max(d.d_inner, nw) * 2 * (d.d_model / 32) + (long long)own_max(d.d_model, nw) * (d.d_inner / 32);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = nw; }
    }
    return best;
}

// Fills every shape / layout field of P (no pointers).  Returns false if the shape does not fit the
// mega path (the chain path then serves it).
inline bool plan(const Dims& d, int G, Params& P)
{
    memset(&P, 0, sizeof P);
    P.L = d.n_layers; P.d_model = d.d_model; P.d_inner = d.d_inner; P.headdim = d.headdim; P.d_state = d.d_state;
    P.ngroups = d.ngroups; P.nheads = d.nheads; P.r = d.r; P.vocab = d.vocab;
    P.gs = d.ngroups * d.d_state;
    P.n_bcdt = 2 * P.gs + d.nheads;
    P.eps = d.eps;
    P.G = G;
    if (G != GRID) return false;
    if (d.d_state % 4 || d.d_model % 32 || d.d_inner % 32 || d.r > 64) return false;
    if (d.d_model > 8192 || d.d_inner > 8192) return false;
    P.NW = pick_workers(d);
    P.NS = G - P.NW;
    P.NT = P.NS - 1;                            // service CTA 0 makes the activation scales, the others hold the row tasks
    P.nch_max = own_max(d.d_inner, P.NW);
    P.nor_max = own_max(d.d_model, P.NW);
    P.r_pad = (d.r + 3) / 4 * 4;
    P.Win = d.d_model / 32;
    P.Wout = d.d_inner / 32;
    P.n_early = P.n_bcdt + d.r;
    if (P.n_early + 1 > NJ_A * THREADS * 4) return false;
    P.tsplit = d.d_inner % 64 == 0 ? 4 : 2;
    P.n_ttask = d.r * P.tsplit;
    if (P.nch_max > 128 || P.nor_max > 128 || d.d_inner < 4 || d.d_model < 4) return false;
    P.ns_sig = dealt(P.n_bcdt, 0, P.NT);
    P.ns_lin = dealt(d.r, 0, P.NT);
    P.ns_tt = dealt(P.n_ttask, 0, P.NT);

    uint32_t off = 0;
    auto take = [&](size_t bytes) { off = up32(off, 16); const uint32_t at = off; off += (uint32_t)bytes; return at; };
    P.c_in_bits = take((size_t)up32(2 * P.nch_max, 4) * P.Win * 4);     // zero rows pad the z | x rows to whole groups of NR_IN
    P.c_out_bits = take((size_t)P.nor_max * P.Wout * 4);
    P.c_in_B = take((size_t)2 * P.nch_max * P.r_pad);
    P.c_out_B = take((size_t)P.nor_max * P.r_pad);
    P.c_in_scale = take((size_t)2 * P.nch_max * 4);
    P.c_in_bs = take((size_t)2 * P.nch_max * 4);
    P.c_out_scale = take((size_t)P.nor_max * 4);
    P.c_out_bs = take((size_t)P.nor_max * 4);
    P.c_conv_w = take((size_t)P.nch_max * 16);
    P.c_conv_b = take((size_t)P.nch_max * 4);
    P.c_alog = take((size_t)P.nch_max * 4);
    P.c_D = take((size_t)P.nch_max * 4);
    P.c_gnorm = take((size_t)P.nch_max * 4);
    P.c_nnorm = take((size_t)P.nor_max * 4);
    P.chunk_bytes = up32(off, 128);

    off = 0;
    P.sc_sign = take((size_t)P.ns_sig * P.Win * 4);
    P.sc_tin = take((size_t)P.ns_lin * d.d_model);
    P.sc_tout = take((size_t)P.ns_tt * (d.d_inner / P.tsplit));
    P.schunk_bytes = up32(off, 128);

    off = 0;
    P.b_eB = take((size_t)P.n_bcdt * P.r_pad);
    P.b_escale = take((size_t)P.n_bcdt * 4);
    P.b_ebs = take((size_t)P.n_bcdt * 4);
    P.b_econv_w = take((size_t)2 * P.gs * 16);
    P.b_econv_b = take((size_t)2 * P.gs * 4);
    P.b_dtb = take((size_t)d.nheads * 4);
    P.b_as_in = take((size_t)P.r_pad * 4);
    P.b_as_out = take((size_t)P.r_pad * 4);
    P.blk_bytes = up32(off, 128);

    P.st_blk = P.chunk_bytes;
    P.st_ssm = P.st_blk + P.blk_bytes;
    P.st_conv = up32(P.st_ssm + (uint32_t)P.nch_max * d.d_state * 4, 128);
    P.st_econv = up32(P.st_conv + (uint32_t)P.nch_max * 16, 128);
    P.stage_bytes = up32(P.st_econv + (uint32_t)P.gs * 32, 128);
    if (P.stage_bytes < P.schunk_bytes) P.stage_bytes = P.schunk_bytes;
    if (P.stage_bytes < 4u * d.d_model) P.stage_bytes = up32(4u * d.d_model, 128);      // an LM item holds >= 4 rows
    P.lm_rows_item = (int)(P.stage_bytes / d.d_model);

    // exchange: part lists of a record's main part and of one small mailbox, 32-bit word offsets, every part 128-byte aligned
    P.u_slot = slot_words(P.nor_max);
    P.g_slot = slot_words(P.nch_max);
    if (P.NW * P.u_slot / 4 > NJ_MAX * THREADS || P.NW * P.g_slot / 4 > NJ_MAX * THREADS) return false;
    if (P.u_slot + P.g_slot > THREADS) return false;
    uint32_t xo = 0;
    auto xtake = [&](size_t words) { xo = up32(xo, 32); const uint32_t at = xo; xo += (uint32_t)words; return at; };
    P.x_U = xtake((size_t)P.NW * P.u_slot);
    P.x_PU = xtake((size_t)2 * P.NW);
    P.x_G = xtake((size_t)P.NW * P.g_slot);
    P.x_PG = xtake((size_t)2 * P.NW);
    P.x_main = up32(xo, 32);
    xo = 0;
    P.x_A = xtake(up32(P.n_early + 1, 4));      // + the scale word(s) made by service CTA 0
    P.x_T = xtake(up32(P.n_ttask, 4) + 8);      // + two scale words, each in a chunk of its own
    P.x_small = up32(xo, 32);

    // shared memory behind the ring
    uint32_t so = 0;
    auto stake = [&](size_t bytes) { so = up32(so, 16); const uint32_t at = so; so += (uint32_t)bytes; return at; };
    const int kmax = d.d_model > d.d_inner ? d.d_model : d.d_inner;
    const uint32_t x_xq = stake(kmax), x_bc = stake((size_t)P.gs * 4), x_cd = stake((size_t)P.gs * 8), x_u = stake((size_t)P.nor_max * 4),
                   x_z = stake((size_t)P.nch_max * 4), x_x = stake((size_t)P.nch_max * 4), x_dt = stake((size_t)d.nheads * 4),
                   x_v = stake((size_t)2 * P.r_pad * 8), x_ea = stake((size_t)P.n_bcdt * 4), x_ai = stake((size_t)up32(2 * P.nch_max, 4) * 4),
                   x_ao = stake((size_t)KS_MAX * P.nor_max * 4), x_chs = stake((size_t)(G + 1) * 4), x_ors = stake((size_t)(G + 1) * 4),
                   x_red = stake(8 * NWARPS), x_slot = stake((size_t)(P.u_slot + P.g_slot) * 4), x_scal = stake(32),
                   x_mbar = stake(8 * MAX_STAGES);
    const uint32_t fixed = up32(so, 128);
    if (fixed + 2 * (size_t)P.stage_bytes > SMEM_LIMIT) return false;
    int stages = (int)((SMEM_LIMIT - fixed) / P.stage_bytes);
    if (stages > MAX_STAGES) stages = MAX_STAGES;
    P.stages = stages;
    const uint32_t ring = (uint32_t)stages * P.stage_bytes;
    P.s_ring = 0;
    P.s_xq = ring + x_xq; P.s_bc = ring + x_bc; P.s_cd = ring + x_cd; P.s_u = ring + x_u; P.s_z = ring + x_z; P.s_x = ring + x_x; P.s_dt = ring + x_dt;
    P.s_v = ring + x_v; P.s_eacc = ring + x_ea; P.s_acc_in = ring + x_ai; P.s_acc_out = ring + x_ao;
    P.s_chs = ring + x_chs; P.s_ors = ring + x_ors; P.s_red = ring + x_red; P.s_slot = ring + x_slot; P.s_scal = ring + x_scal;
    P.s_mbar = ring + x_mbar;
    P.smem_bytes = ring + fixed;
    return true;
}

// arena regions of the mega path (byte sizes)
struct Regions {
    size_t chunks, schunks, blocks, xbuf, am;
};
inline Regions regions(const Params& P)
{
    Regions r;
    const size_t nl = (size_t)(P.L > 0 ? P.L : 1);
    r.chunks = nl * P.NW * P.chunk_bytes;
    r.schunks = nl * P.NT * P.schunk_bytes;
    r.blocks = nl * P.blk_bytes;
    r.xbuf = (size_t)2 * nl * ((size_t)P.x_main + (size_t)MBOX * P.x_small) * 4;      // 2 sets x L records
    r.am = (size_t)P.G * 8 + 64;
    return r;
}

inline float half_bits_to_float(uint16_t h)     // exact binary16 -> binary32 (host; own code)
{
    const uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
    const uint32_t e = (h >> 10) & 0x1fu, m = h & 0x3ffu;
    uint32_t bits;
    if (e == 0) {
        if (m == 0) bits = sign;
        else {                                   // subnormal: normalise
            int sh = 0;
            uint32_t mm = m;
            while (!(mm & 0x400u)) { mm <<= 1; ++sh; }
            bits = sign | ((uint32_t)(127 - 15 - sh + 1) << 23) | ((mm & 0x3ffu) << 13);
        }
    } else if (e == 31) bits = sign | 0x7f800000u | (m << 13);
    else bits = sign | ((e - 15 + 127) << 23) | (m << 13);
    float f;
    memcpy(&f, &bits, 4);
    return f;
}

inline int plane_pos_host(int k, int K)
{
    return ((k & 16) ? (K >> 1) : 0) + ((k >> 5) << 4) + (k & 15);
}

// canonical sign word (bit p = element p of the 32-block) -> kernel sign word (bit 8j + i = element 4i + j)
inline uint32_t permute_sign_word(uint32_t w)
{
    uint32_t o = 0;
    for (int p = 0; p < 32; ++p)
        if ((w >> p) & 1u) o |= 1u << (8 * (p & 3) + (p >> 2));
    return o;
}
struct SignLut {
    uint32_t t[4][256];
    SignLut()
    {
        for (int b = 0; b < 4; ++b)
            for (int v = 0; v < 256; ++v) t[b][v] = permute_sign_word((uint32_t)v << (8 * b));
    }
    uint32_t operator()(uint32_t w) const { return t[0][w & 255u] | t[1][(w >> 8) & 255u] | t[2][(w >> 16) & 255u] | t[3][w >> 24]; }
};
inline void copy_sign_row(uint32_t* dst, const uint32_t* src, int W)
{
    static const SignLut lut;
    for (int w = 0; w < W; ++w) dst[w] = lut(src[w]);
}

// host pointers to one layer of the canonical blob
struct HostLayer {
    const float* norm_w;
    const uint32_t* in_sign; const uint16_t* in_row_scale;
    const int8_t* in_A; const float* in_a_s; const int8_t* in_B; const float* in_b_s;
    const float* conv_w; const float* conv_b;
    const float* A_log; const float* dt_bias; const float* D;
    const float* gnorm_w;
    const uint32_t* out_sign; const uint16_t* out_row_scale;
    const int8_t* out_A; const float* out_a_s; const int8_t* out_B; const float* out_b_s;
};

// chunk of (layer, worker c): `next_norm_w` is the norm weight applied to u after this layer
inline void pack_chunk(const Params& P, const HostLayer& H, const float* next_norm_w, int c, uint8_t* out)
{
    memset(out, 0, P.chunk_bytes);
    const int ch0 = own_start(c, P.d_inner, P.NW), nch = own_start(c + 1, P.d_inner, P.NW) - ch0;
    const int or0 = own_start(c, P.d_model, P.NW), nor = own_start(c + 1, P.d_model, P.NW) - or0;
    auto put_in_row = [&](int slot, int row) {
        copy_sign_row((uint32_t*)(out + P.c_in_bits + (size_t)slot * P.Win * 4), H.in_sign + (size_t)row * P.Win, P.Win);
        memcpy(out + P.c_in_B + (size_t)slot * P.r_pad, H.in_B + (size_t)row * P.r, P.r);
        ((float*)(out + P.c_in_scale))[slot] = half_bits_to_float(H.in_row_scale[row]);
        ((float*)(out + P.c_in_bs))[slot] = H.in_b_s[row];
    };
    for (int i = 0; i < nch; ++i) {
        const int ch = ch0 + i, h = ch / P.headdim;
        put_in_row(i, ch);                                   // z row
        put_in_row(nch + i, P.d_inner + ch);                 // x row
        memcpy(out + P.c_conv_w + 16 * (size_t)i, H.conv_w + 4 * (size_t)ch, 16);
        ((float*)(out + P.c_conv_b))[i] = H.conv_b[ch];
        ((float*)(out + P.c_alog))[i] = H.A_log[h];
        ((float*)(out + P.c_D))[i] = H.D[h];
        ((float*)(out + P.c_gnorm))[i] = H.gnorm_w[ch];
    }
    for (int i = 0; i < nor; ++i) {
        const int row = or0 + i;
        copy_sign_row((uint32_t*)(out + P.c_out_bits + (size_t)i * P.Wout * 4), H.out_sign + (size_t)row * P.Wout, P.Wout);
        memcpy(out + P.c_out_B + (size_t)i * P.r_pad, H.out_B + (size_t)row * P.r, P.r);
        ((float*)(out + P.c_out_scale))[i] = half_bits_to_float(H.out_row_scale[row]);
        ((float*)(out + P.c_out_bs))[i] = H.out_b_s[row];
        ((float*)(out + P.c_nnorm))[i] = next_norm_w[row];
    }
}

inline void permute_row(const int8_t* A, int K, int8_t* out)
{
    for (int k = 0; k < K; ++k) out[plane_pos_host(k, K)] = A[k];
}

// chunk of (layer, task CTA s): the B|C|dt sign rows s, s + NT, ..., the in_proj LoRA-down rows s, s + NT, ... and the
// out_proj LoRA-down partial tasks s, s + NT, ... (task q = row q / tsplit, part q % tsplit of the plane-permuted row)
inline void pack_schunk(const Params& P, const HostLayer& H, int s, uint8_t* out, std::vector<int8_t>& tmp)
{
    memset(out, 0, P.schunk_bytes);
    for (int k = 0, e = s; e < P.n_bcdt; ++k, e += P.NT)
        copy_sign_row((uint32_t*)(out + P.sc_sign + (size_t)k * P.Win * 4), H.in_sign + (size_t)(2 * P.d_inner + e) * P.Win, P.Win);
    for (int k = 0, j = s; j < P.r; ++k, j += P.NT)
        permute_row(H.in_A + (size_t)j * P.d_model, P.d_model, (int8_t*)(out + P.sc_tin + (size_t)k * P.d_model));
    const int tbytes = P.d_inner / P.tsplit;
    tmp.resize((size_t)P.d_inner);
    for (int k = 0, q = s; q < P.n_ttask; ++k, q += P.NT) {
        permute_row(H.out_A + (size_t)(q / P.tsplit) * P.d_inner, P.d_inner, tmp.data());
        memcpy(out + P.sc_tout + (size_t)k * tbytes, tmp.data() + (size_t)(q % P.tsplit) * tbytes, tbytes);
    }
}

// block of a layer: what every CTA needs to finish the B | C | dt rows itself
inline void pack_block(const Params& P, const HostLayer& H, uint8_t* out)
{
    memset(out, 0, P.blk_bytes);
    for (int e = 0; e < P.n_bcdt; ++e) {
        const int row = 2 * P.d_inner + e;
        {   // word-major: word g of row e (its LoRA-up bytes 4g .. 4g+3, zero padded) at [g][e]
            uint8_t rowb[64] = { 0 };
            memcpy(rowb, H.in_B + (size_t)row * P.r, P.r);
            for (int g = 0; g < P.r_pad / 4; ++g) memcpy(out + P.b_eB + ((size_t)g * P.n_bcdt + e) * 4, rowb + 4 * g, 4);
        }
        ((float*)(out + P.b_escale))[e] = half_bits_to_float(H.in_row_scale[row]);
        ((float*)(out + P.b_ebs))[e] = H.in_b_s[row];
        if (e < 2 * P.gs) {
            memcpy(out + P.b_econv_w + 16 * (size_t)e, H.conv_w + 4 * (size_t)(P.d_inner + e), 16);
            ((float*)(out + P.b_econv_b))[e] = H.conv_b[P.d_inner + e];
        } else {
            ((float*)(out + P.b_dtb))[e - 2 * P.gs] = H.dt_bias[e - 2 * P.gs];
        }
    }
    for (int j = 0; j < P.r; ++j) {
        ((float*)(out + P.b_as_in))[j] = H.in_a_s[j];
        ((float*)(out + P.b_as_out))[j] = H.out_a_s[j];
    }
}

}  // namespace mega
}  // namespace dfssm

namespace dfssm {
namespace mega {

// the shapes of BASELINE.json's configs get a kernel with compile-time dimensions; any other shape uses the run-time-shape
// kernel (with the taps / profiler code compiled in only when asked for)
using Shape0 = ShapeCT<256, 512, 64, 64, 1, 8>;
using Shape1 = ShapeCT<768, 1536, 64, 128, 1, 16>;
using Shape2 = ShapeCT<2048, 4096, 64, 128, 1, 32>;
using Shape4 = ShapeCT<2560, 5120, 64, 128, 1, 32>;

template <class S>
inline bool shape_is(const Dims& d)
{
    return d.d_model == S::d_model && d.d_inner == S::d_inner && d.headdim == S::headdim && d.d_state == S::d_state &&
           d.ngroups == S::ngroups && d.r == S::r;
}

typedef void (*KernelFn)(const Params);
inline KernelFn pick_kernel(const Dims& d, bool taps, bool prof)
{
    if (!taps) {
        if (shape_is<Shape0>(d)) return prof ? k_mega<Shape0, false, true> : k_mega<Shape0, false, false>;
        if (shape_is<Shape1>(d)) return prof ? k_mega<Shape1, false, true> : k_mega<Shape1, false, false>;
        if (shape_is<Shape2>(d)) return prof ? k_mega<Shape2, false, true> : k_mega<Shape2, false, false>;
        if (shape_is<Shape4>(d)) return prof ? k_mega<Shape4, false, true> : k_mega<Shape4, false, false>;
    }
    if (taps || prof) return k_mega<ShapeRT, true, true>;
    return k_mega<ShapeRT, false, false>;
}

}  // namespace mega
}  // namespace dfssm
