// Host side of the mega path: the per-(layer, CTA) chunk layout, the shared-memory plan, and the
// load-time repack of the canonical blob (DESIGN.md sections 3 and 6) into that layout.
#pragma once
#include <cstring>
#include <vector>

#include "dfssm_mega.cuh"

namespace dfssm {
namespace mega {

constexpr int GRID = 148;                       // one CTA per B200 SM
constexpr size_t SMEM_LIMIT = 232448 - 1024;    // 227 KB opt-in maximum minus the kernel's static shared memory

inline uint32_t up32(uint32_t x, uint32_t a) { return (x + a - 1) / a * a; }

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
    if (d.d_state % 4 || d.d_model % 32 || d.d_inner % 32 || d.r > 64) return false;
    P.nch_max = (d.d_inner + G - 1) / G;
    P.nor_max = (d.d_model + G - 1) / G;
    P.nb_max = (P.n_bcdt + G - 1) / G;
    P.n_slots = 2 * P.nch_max + P.nb_max;
    P.r_pad = (d.r + 3) / 4 * 4;
    P.Win = d.d_model / 32;
    P.Wout = d.d_inner / 32;
    P.wpc1 = (P.nor_max + CODES_PER_WORD - 1) / CODES_PER_WORD;
    P.wpc3 = (P.nch_max + CODES_PER_WORD - 1) / CODES_PER_WORD;
    if (P.wpc1 > THREADS || P.wpc3 > THREADS) return false;

    uint32_t off = 0;
    auto take = [&](size_t bytes) { off = up32(off, 16); const uint32_t at = off; off += (uint32_t)bytes; return at; };
    P.c_in_bits = take((size_t)P.n_slots * P.Win * 4);
    P.c_out_bits = take((size_t)P.nor_max * P.Wout * 4);
    P.c_in_B = take((size_t)P.n_slots * P.r_pad);
    P.c_out_B = take((size_t)P.nor_max * P.r_pad);
    P.c_in_scale = take((size_t)P.n_slots * 4);
    P.c_in_bs = take((size_t)P.n_slots * 4);
    P.c_out_scale = take((size_t)P.nor_max * 4);
    P.c_out_bs = take((size_t)P.nor_max * 4);
    P.c_conv_w = take((size_t)P.nch_max * 16);
    P.c_conv_b = take((size_t)P.nch_max * 4);
    P.c_e_conv_w = take((size_t)P.nb_max * 16);
    P.c_e_conv_b = take((size_t)P.nb_max * 4);
    P.c_e_dtb = take((size_t)P.nb_max * 4);
    P.c_alog = take((size_t)P.nch_max * 4);
    P.c_D = take((size_t)P.nch_max * 4);
    P.c_gnorm = take((size_t)P.nch_max * 4);
    P.c_nnorm = take((size_t)P.nor_max * 4);
    P.c_as_in = take((size_t)P.r_pad * 4);
    P.c_as_out = take((size_t)P.r_pad * 4);
    P.chunk_bytes = up32(off, 128);

    P.st_ssm = P.chunk_bytes;
    P.st_conv = up32(P.st_ssm + (uint32_t)P.nch_max * d.d_state * 4, 128);
    P.stage_bytes = up32(P.st_conv + (uint32_t)P.nch_max * 16, 128);
    if (P.stage_bytes < 4u * d.d_model) P.stage_bytes = up32(4u * d.d_model, 128);      // an LM item holds >= 4 rows
    P.lm_rows_item = (int)(P.stage_bytes / d.d_model);

    // shared memory behind the ring
    uint32_t so = 0;
    auto stake = [&](size_t bytes) { so = up32(so, 16); const uint32_t at = so; so += (uint32_t)bytes; return at; };
    const int kmax = d.d_model > d.d_inner ? d.d_model : d.d_inner;
    const int nmax = P.nch_max > P.nor_max ? P.nch_max : P.nor_max;
    const uint32_t x_xq = stake(kmax), x_bc = stake((size_t)P.n_bcdt * 4), x_u = stake((size_t)P.nor_max * 4),
                   x_z = stake((size_t)P.nch_max * 4), x_x = stake((size_t)P.nch_max * 4), x_tq = stake((size_t)nmax * 4),
                   x_vin = stake((size_t)P.r_pad * 4), x_vout = stake((size_t)P.r_pad * 4), x_ai = stake((size_t)P.n_slots * 4),
                   x_ao = stake((size_t)P.nor_max * 4), x_chs = stake((size_t)(G + 1) * 4), x_ors = stake((size_t)(G + 1) * 4),
                   x_stats = stake((size_t)3 * G * 4), x_red = stake(256), x_mbar = stake(8 * MAX_STAGES);
    const uint32_t fixed = up32(so, 128);
    if (fixed + 2 * (size_t)P.stage_bytes > SMEM_LIMIT) return false;
    int stages = (int)((SMEM_LIMIT - fixed) / P.stage_bytes);
    if (stages > MAX_STAGES) stages = MAX_STAGES;
    P.stages = stages;
    const uint32_t ring = (uint32_t)stages * P.stage_bytes;
    P.s_ring = 0;
    P.s_xq = ring + x_xq; P.s_bc = ring + x_bc; P.s_u = ring + x_u; P.s_z = ring + x_z; P.s_x = ring + x_x;
    P.s_tq = ring + x_tq; P.s_vin = ring + x_vin; P.s_vout = ring + x_vout; P.s_acc_in = ring + x_ai;
    P.s_acc_out = ring + x_ao; P.s_chs = ring + x_chs; P.s_ors = ring + x_ors; P.s_stats = ring + x_stats;
    P.s_red = ring + x_red; P.s_mbar = ring + x_mbar;
    P.smem_bytes = ring + fixed;
    return true;
}

// arena regions of the mega path (byte sizes)
struct Regions {
    size_t chunks, A_in, A_out, xbuf, am;
};
inline Regions regions(const Params& P)
{
    Regions r;
    r.chunks = (size_t)(P.L > 0 ? P.L : 1) * P.G * P.chunk_bytes;
    r.A_in = (size_t)(P.L > 0 ? P.L : 1) * P.r * P.d_model;
    r.A_out = (size_t)(P.L > 0 ? P.L : 1) * P.r * P.d_inner;
    // exchange words: stats x2 (3G each), codes (G*wpc1, G*wpc3), t x2 (64 each), bc (n_bcdt)
    r.xbuf = 8 * ((size_t)6 * P.G + (size_t)P.G * (P.wpc1 + P.wpc3) + 128 + P.n_bcdt + 64);
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
    const int w = k >> 5, p = k & 31, j = p >> 3, i = p & 7;
    return (i < 4 ? 0 : (K >> 1)) + 16 * w + 4 * (i & 3) + j;
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

// chunk of (layer, CTA c): `next_norm_w` is the norm weight applied to u after this layer
inline void pack_chunk(const Params& P, const HostLayer& H, const float* next_norm_w, int c, uint8_t* out)
{
    memset(out, 0, P.chunk_bytes);
    const int G = P.G;
    const int ch0 = (int)(((long long)c * P.d_inner) / G), nch = (int)(((long long)(c + 1) * P.d_inner) / G) - ch0;
    const int or0 = (int)(((long long)c * P.d_model) / G), nor = (int)(((long long)(c + 1) * P.d_model) / G) - or0;
    auto put_in_row = [&](int slot, int row) {
        memcpy(out + P.c_in_bits + (size_t)slot * P.Win * 4, H.in_sign + (size_t)row * P.Win, (size_t)P.Win * 4);
        memcpy(out + P.c_in_B + (size_t)slot * P.r_pad, H.in_B + (size_t)row * P.r, P.r);
        ((float*)(out + P.c_in_scale))[slot] = half_bits_to_float(H.in_row_scale[row]);
        ((float*)(out + P.c_in_bs))[slot] = H.in_b_s[row];
    };
    for (int i = 0; i < nch; ++i) {
        const int ch = ch0 + i, h = ch / P.headdim;
        put_in_row(i, ch);                                   // z row
        put_in_row(P.nch_max + i, P.d_inner + ch);           // x row
        memcpy(out + P.c_conv_w + 16 * (size_t)i, H.conv_w + 4 * (size_t)ch, 16);
        ((float*)(out + P.c_conv_b))[i] = H.conv_b[ch];
        ((float*)(out + P.c_alog))[i] = H.A_log[h];
        ((float*)(out + P.c_D))[i] = H.D[h];
        ((float*)(out + P.c_gnorm))[i] = H.gnorm_w[ch];
    }
    for (int k = 0, e = c; e < P.n_bcdt; ++k, e += G) {      // early rows: B | C | dt
        put_in_row(2 * P.nch_max + k, 2 * P.d_inner + e);
        if (e < 2 * P.gs) {
            memcpy(out + P.c_e_conv_w + 16 * (size_t)k, H.conv_w + 4 * (size_t)(P.d_inner + e), 16);
            ((float*)(out + P.c_e_conv_b))[k] = H.conv_b[P.d_inner + e];
        } else {
            ((float*)(out + P.c_e_dtb))[k] = H.dt_bias[e - 2 * P.gs];
        }
    }
    for (int i = 0; i < nor; ++i) {
        const int row = or0 + i;
        memcpy(out + P.c_out_bits + (size_t)i * P.Wout * 4, H.out_sign + (size_t)row * P.Wout, (size_t)P.Wout * 4);
        memcpy(out + P.c_out_B + (size_t)i * P.r_pad, H.out_B + (size_t)row * P.r, P.r);
        ((float*)(out + P.c_out_scale))[i] = half_bits_to_float(H.out_row_scale[row]);
        ((float*)(out + P.c_out_bs))[i] = H.out_b_s[row];
        ((float*)(out + P.c_nnorm))[i] = next_norm_w[row];
    }
    for (int j = 0; j < P.r; ++j) {
        ((float*)(out + P.c_as_in))[j] = H.in_a_s[j];
        ((float*)(out + P.c_as_out))[j] = H.out_a_s[j];
    }
}

inline void permute_A(const int8_t* A, int r, int K, int8_t* out)
{
    for (int j = 0; j < r; ++j)
        for (int k = 0; k < K; ++k) out[(size_t)j * K + plane_pos_host(k, K)] = A[(size_t)j * K + k];
}

}  // namespace mega
}  // namespace dfssm
