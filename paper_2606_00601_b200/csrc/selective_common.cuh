// selective_common.cuh — pieces shared by the selective_scan_fwd kernels: packed fp32x2
// arithmetic, 2^x on the fma pipe, and the optional fused steps either side of the scan
// (P:284): softplus/bias prologue, silu(z) gate, resets.
#pragma once

#include "common.cuh"

namespace affinescan {

constexpr float kLn2 = 0.6931471805599453f;

// ------------------------------------------------------------------ optional fused steps
// All pointers may be NULL.  When every field is NULL/0 the kernels take the plain path.
struct SelectiveExt {
    const void* z;              // [batch, d_inner, L] io dtype: y <- y * silu(z)
    const float* delta_bias;    // [d_inner]: Delta = delta + bias[d]
    const unsigned char* reset; // [batch, L]: nonzero = step t starts a new sequence (h_{t-1} := 0)
    int delta_softplus;         // Delta = softplus(delta + bias)
};

__device__ __forceinline__ float lg2_approx(float x)
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// softplus(v) = log(1 + e^v) = max(v, 0) + log1p(e), e = 2^(-|v| log2 e) in (0, 1]: MUFU.EX2 +
// MUFU.LG2 and a few fp32 ops, finite for every v.  For small e (|v| > 4.6) log1p(e) is taken
// from its series e - e^2/2 + e^3/3 instead of log2(1 + e), so that a tiny Delta = e^v keeps its
// full relative accuracy (a slow channel's memory is 1/(Delta |A|)).
__device__ __forceinline__ float softplus_f(float v)
{
    const float e = ex2_approx(-fabsf(v) * kLog2e);
    const float series = e * fmaf(e, fmaf(e, 0.33333334f, -0.5f), 1.0f);
    const float l1p = e < 0.01f ? series : lg2_approx(1.0f + e) * kLn2;
    return fmaxf(v, 0.0f) + l1p;
}
// silu(v) = v / (1 + e^-v): MUFU.EX2 + MUFU.RCP (relative error ~1e-6).
__device__ __forceinline__ float silu_f(float v)
{
    return v * rcp_approx(1.0f + ex2_approx(-v * kLog2e));
}
// silu(v) = (v/2) (1 + tanh(v/2)) with ONE MUFU.TANH (relative error ~5e-4): used for bf16
// outputs only, whose own rounding is 2e-3.
__device__ __forceinline__ float silu_tanh_f(float v)
{
    const float hv = 0.5f * v;
    float t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(hv));
    return fmaf(t, hv, hv);
}
template <typename T>
__device__ __forceinline__ float silu_io(float v)
{
    return sizeof(T) == 2 ? silu_tanh_f(v) : silu_f(v);
}

// ------------------------------------------------------------------ packed fp32x2 arithmetic
// A "pair" is two fp32 values in one 64-bit register pair; SASS: FFMA2 / FMUL2.
using pair_t = unsigned long long;

__device__ __forceinline__ pair_t pk(float lo, float hi)
{
    pair_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(pair_t v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ pair_t fma2(pair_t a, pair_t b, pair_t c)
{
    pair_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ pair_t mul2(pair_t a, pair_t b)
{
    pair_t d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// ------------------------------------------------------------------ 2^x on the fma pipe
// x = i + r, i = round(x), r in [-1/2, 1/2];  2^x = 2^i * p(r),  p(r) = 1 + r*q(r) with q the
// minimax approximation of (2^r - 1)/r (error measured relative to 2^r - 1, so that a = 2^x close
// to 1 keeps an accurate 1 - a: DESIGN.md §7).  Valid for |x| <= 126 (the caller checks delta).
template <int DEG>
struct Exp2Coef;
template <>
struct Exp2Coef<3> {  // max |p - 2^r| / |2^r - 1| = 4.3e-4
    static __device__ __forceinline__ float c(int i)
    {
        constexpr float k[3] = {6.931782961e-01f, 2.420288622e-01f, 5.550396442e-02f};
        return k[i];
    }
};
template <>
struct Exp2Coef<5> {  // 4.3e-7 (then fp32 rounding)
    static __device__ __forceinline__ float c(int i)
    {
        constexpr float k[5] = {6.931471229e-01f, 2.402235121e-01f, 5.550500378e-02f,
                                9.666245431e-03f, 1.333353925e-03f};
        return k[i];
    }
};

// {2^(d*A2.lo), 2^(d*A2.hi)} for dd = {d,d}: 3 + DEG FFMA2 and two integer shift-adds.
template <int DEG>
__device__ __forceinline__ pair_t exp2_poly2(pair_t dd, pair_t A2p)
{
    constexpr float kMagic = 12582912.0f;  // 1.5 * 2^23: fma rounds x to the nearest integer
    const pair_t magic = pk(kMagic, kMagic);
    const pair_t t = fma2(dd, A2p, magic);                   // bits(t) = 0x4B400000 + i
    const pair_t ni = fma2(t, pk(-1.0f, -1.0f), magic);      // -i, exact
    const pair_t r = fma2(dd, A2p, ni);                      // x - i with one rounding
    pair_t q = pk(Exp2Coef<DEG>::c(DEG - 1), Exp2Coef<DEG>::c(DEG - 1));
#pragma unroll
    for (int j = DEG - 2; j >= 0; --j) q = fma2(q, r, pk(Exp2Coef<DEG>::c(j), Exp2Coef<DEG>::c(j)));
    const pair_t p = fma2(q, r, pk(1.0f, 1.0f));
    float plo, phi, tlo, thi;
    upk(p, plo, phi);
    upk(t, tlo, thi);
    // 2^i by adding i to the exponent field: (bits(t) << 23) == i << 23 (mod 2^32)
    const float alo = __uint_as_float(__float_as_uint(plo) + (__float_as_uint(tlo) << 23));
    const float ahi = __uint_as_float(__float_as_uint(phi) + (__float_as_uint(thi) << 23));
    return pk(alo, ahi);
}

}  // namespace affinescan
