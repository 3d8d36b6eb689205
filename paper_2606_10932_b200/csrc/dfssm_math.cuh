// Device arithmetic of the DF-SSM decode step ("arithmetic contract").
//
// Every elementwise float operation is ONE IEEE binary32 round-to-nearest-even operation,
// spelled with an explicit intrinsic so the compiler can neither contract nor reassociate it;
// subnormals are kept (the library is built without -ftz / --use_fast_math, with -fmad=false).
// Reductions accumulate in binary64 from exact binary32 x binary32 products and round once.
// exp / log1p / softplus / SiLU are the fixed operation sequences of DESIGN.md section 5.4.
#pragma once
#include <cuda_fp16.h>
#include <stdint.h>

namespace dfssm {

__device__ __forceinline__ float fmul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float fadd(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float ffma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ float fdiv(float a, float b) { return __fdiv_rn(a, b); }

// exp(x): clamp to [-87, 88] (x < -87 -> 0); n = rint(x*log2 e);
// r = x - n*ln2 by a two-constant Cody-Waite reduction with fma; degree-7 Taylor polynomial
// (coefficients 1/k! rounded to binary32) in Horner form; multiply by 2^n built in the exponent field.
__device__ __forceinline__ float sp_expf(float x)
{
    if (x < -87.0f) return 0.0f;
    if (x > 88.0f) x = 88.0f;
    const float nr = fadd(fmul(x, 0x1.715476p+0f), 12582912.0f);    // rint by magic-number addition (|n| <= 127)
    const float n = fadd(nr, -12582912.0f);
    float r = ffma(n, -0x1.63p-1f, x);
    r = ffma(n, 0x1.bd0106p-13f, r);               // -LN2_LO with LN2_LO = -0x1.bd0106p-13
    float p = 0x1.a01a02p-13f;                     // 1/7!
    p = ffma(p, r, 0x1.6c16c2p-10f);               // 1/6!
    p = ffma(p, r, 0x1.111112p-7f);                // 1/5!
    p = ffma(p, r, 0x1.555556p-5f);                // 1/4!
    p = ffma(p, r, 0x1.555556p-3f);                // 1/3!
    p = ffma(p, r, 0x1p-1f);                       // 1/2!
    p = ffma(p, r, 1.0f);
    p = ffma(p, r, 1.0f);
    const int ni = __float_as_int(nr) - 0x4b400000;   // in [-126, 127]
    return fmul(p, __uint_as_float((uint32_t)(ni + 127) << 23));
}

// log(1+t), t in [0,1]: s = t/(2+t); 2*s*(1 + s^2/3 + ... + s^16/17)
__device__ __forceinline__ float sp_log1pf(float t)
{
    const float s = fdiv(t, fadd(2.0f, t));
    const float s2 = fmul(s, s);
    float p = 0x1.e1e1e2p-5f;                      // 1/17
    p = ffma(p, s2, 0x1.111112p-4f);               // 1/15
    p = ffma(p, s2, 0x1.3b13b2p-4f);               // 1/13
    p = ffma(p, s2, 0x1.745d18p-4f);               // 1/11
    p = ffma(p, s2, 0x1.c71c72p-4f);               // 1/9
    p = ffma(p, s2, 0x1.24924ap-3f);               // 1/7
    p = ffma(p, s2, 0x1.99999ap-3f);               // 1/5
    p = ffma(p, s2, 0x1.555556p-2f);               // 1/3
    p = ffma(p, s2, 1.0f);
    return fmul(2.0f, fmul(s, p));
}

// softplus(x) = max(x,0) + log1p(exp(-|x|)); x for x > 20
__device__ __forceinline__ float sp_softplusf(float x)
{
    if (x > 20.0f) return x;
    const float e = sp_expf(-fabsf(x));
    const float l = sp_log1pf(e);
    const float m = x > 0.0f ? x : 0.0f;
    return fadd(m, l);
}

// SiLU(x) = x / (1 + exp(-x))
__device__ __forceinline__ float siluf(float x)
{
    return fdiv(x, fadd(1.0f, sp_expf(-x)));
}

// exact product of two binary32 values accumulated in binary64: a + (double)x*(double)y.
// The product has at most 48 significant bits, so the fused and the unfused forms agree.
__device__ __forceinline__ double dacc(double a, float x, float y)
{
    return __fma_rn((double)x, (double)y, a);
}

// dp4a with UNSIGNED bytes in a and SIGNED bytes in b: c + sum_j a.u8[j] * b.s8[j]
__device__ __forceinline__ int dp4a_us(uint32_t a, int b, int c)
{
    int d;
    asm("dp4a.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
// signed x signed
__device__ __forceinline__ int dp4a_ss(int a, int b, int c) { return __dp4a(a, b, c); }

// per-token absmax quantiser (R4): codes from t = v*w, inv = 127/amax, ties to even, clamp +-127.
// rint by the magic-number addition (exact ties-to-even for |x| < 2^22); the FRND / F2I conversions run at a
// quarter of the fp32 rate and the quantiser is on the critical path.  The clamp of R4 can never act here:
// |t| <= amax and inv = fl(127/amax) give |fl(t*inv)| <= 127 (1 + 2^-23), which rounds to 127.
__device__ __forceinline__ int quant_code(float t, float inv)
{
    const float r = fadd(fmul(t, inv), 12582912.0f);            // 1.5 * 2^23
    return __float_as_int(r) - 0x4b400000;
}

// ---- warp / block reductions (any tree is allowed: sums are binary64, max is exact) ----
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// sum over the lanes {k, k + stride, k + 2 stride, ...} (stride a power of two; the other lanes hold 0): the result is
// valid in those lanes.  Saves log2(stride) of the five fp64 shuffle steps when only every stride-th lane has a value.
__device__ __forceinline__ double warp_sum_strided(double v, int stride)
{
    for (int o = stride; o < 32; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// max of NON-NEGATIVE floats (all uses: |x| maxima): their bit patterns order like unsigned integers, so one REDUX does it
__device__ __forceinline__ float warp_max(float v)
{
    return __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(v)));
}
__device__ __forceinline__ int warp_sum_i(int v)
{
    return __reduce_add_sync(0xffffffffu, v);
}

}  // namespace dfssm
