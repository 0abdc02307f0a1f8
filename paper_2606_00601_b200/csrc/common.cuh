// common.cuh — device helpers shared by the libaffinescan kernels (sm_100a).
//
// P:<n> = /root/reference/PAPER.md line n; BJ = BASELINE.json north_star.
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace affinescan {

constexpr unsigned kFullMask = 0xffffffffu;
constexpr float kLog2e = 1.4426950408889634f;

// Affine transition pair (A_t, U_t) = (a_t, b_t x_t), Eq.(6).
struct Pair {
    float P;  // multiplicative part A
    float U;  // additive part U
};

__device__ __forceinline__ Pair identity_pair() { return Pair{1.0f, 0.0f}; }

// (A2,U2) (+) (A1,U1) = (A2*A1, A2*U1 + U2), Eq.(7).  `later` is the LEFT operand.
__device__ __forceinline__ Pair compose(Pair later, Pair earlier)
{
    return Pair{later.P * earlier.P, fmaf(later.P, earlier.U, later.U)};
}

// h' = A*h + U : apply a (composed) transition to a state.
__device__ __forceinline__ float apply(Pair e, float h) { return fmaf(e.P, h, e.U); }

// 2^x on the SFU: exactly one MUFU.EX2 (Q11).
__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ Pair shfl_up_pair(Pair v, int delta)
{
    return Pair{__shfl_up_sync(kFullMask, v.P, delta), __shfl_up_sync(kFullMask, v.U, delta)};
}
__device__ __forceinline__ Pair shfl_down_pair(Pair v, int delta)
{
    return Pair{__shfl_down_sync(kFullMask, v.P, delta), __shfl_down_sync(kFullMask, v.U, delta)};
}
__device__ __forceinline__ Pair shfl_pair(Pair v, int src)
{
    return Pair{__shfl_sync(kFullMask, v.P, src), __shfl_sync(kFullMask, v.U, src)};
}

// Inclusive Kogge–Stone scan of pairs across the 32 lanes; lane i ends with
// e_i (+) e_{i-1} (+) ... (+) e_0 (lane 0 = earliest).
__device__ __forceinline__ Pair warp_inclusive_scan(Pair v, int lane)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const Pair prev = shfl_up_pair(v, d);
        if (lane >= d) v = compose(v, prev);
    }
    return v;
}

// ------------------------------------------------------------------ io dtype traits
template <typename T>
struct Io;

template <>
struct Io<float> {
    static constexpr int kVec = 4;  // elements per 128-bit access
};
template <>
struct Io<__nv_bfloat16> {
    static constexpr int kVec = 8;
};

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi)
{
    const __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);  // RNE, one F2FP
    return *reinterpret_cast<const uint32_t*>(&v);
}

// 128 bits of io-dtype storage -> Io<T>::kVec floats (exact widening).
template <typename T>
__device__ __forceinline__ void unpack128(const uint4& w, float (&v)[Io<T>::kVec]);
template <>
__device__ __forceinline__ void unpack128<float>(const uint4& w, float (&v)[4])
{
    v[0] = __uint_as_float(w.x); v[1] = __uint_as_float(w.y);
    v[2] = __uint_as_float(w.z); v[3] = __uint_as_float(w.w);
}
template <>
__device__ __forceinline__ void unpack128<__nv_bfloat16>(const uint4& w, float (&v)[8])
{
    v[0] = bf16_lo(w.x); v[1] = bf16_hi(w.x);
    v[2] = bf16_lo(w.y); v[3] = bf16_hi(w.y);
    v[4] = bf16_lo(w.z); v[5] = bf16_hi(w.z);
    v[6] = bf16_lo(w.w); v[7] = bf16_hi(w.w);
}

// Access<T, VEC, kStream>: VEC == Io<T>::kVec -> one 128-bit access (p must be 16-byte aligned),
// VEC == 1 -> one scalar access.  kStream selects the streaming (evict-first) policy.
template <typename T, int VEC, bool kStream>
struct Access;

template <bool kStream>
struct Access<float, 4, kStream> {
    static __device__ __forceinline__ void load(const float* p, float (&v)[4])
    {
        const float4 r = kStream ? __ldcs(reinterpret_cast<const float4*>(p))
                                 : __ldg(reinterpret_cast<const float4*>(p));
        v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w;
    }
    static __device__ __forceinline__ void store(float* p, const float (&v)[4])
    {
        const float4 r = make_float4(v[0], v[1], v[2], v[3]);
        if (kStream) __stcs(reinterpret_cast<float4*>(p), r);
        else *reinterpret_cast<float4*>(p) = r;
    }
};

template <bool kStream>
struct Access<float, 1, kStream> {
    static __device__ __forceinline__ void load(const float* p, float (&v)[1])
    {
        v[0] = kStream ? __ldcs(p) : __ldg(p);
    }
    static __device__ __forceinline__ void store(float* p, const float (&v)[1])
    {
        if (kStream) __stcs(p, v[0]);
        else *p = v[0];
    }
};

template <bool kStream>
struct Access<__nv_bfloat16, 8, kStream> {
    static __device__ __forceinline__ void load(const __nv_bfloat16* p, float (&v)[8])
    {
        const uint4 r = kStream ? __ldcs(reinterpret_cast<const uint4*>(p))
                                : __ldg(reinterpret_cast<const uint4*>(p));
        v[0] = bf16_lo(r.x); v[1] = bf16_hi(r.x);
        v[2] = bf16_lo(r.y); v[3] = bf16_hi(r.y);
        v[4] = bf16_lo(r.z); v[5] = bf16_hi(r.z);
        v[6] = bf16_lo(r.w); v[7] = bf16_hi(r.w);
    }
    static __device__ __forceinline__ void store(__nv_bfloat16* p, const float (&v)[8])
    {
        const uint4 r = make_uint4(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3]),
                                   pack_bf16x2(v[4], v[5]), pack_bf16x2(v[6], v[7]));
        if (kStream) __stcs(reinterpret_cast<uint4*>(p), r);
        else *reinterpret_cast<uint4*>(p) = r;
    }
};

template <bool kStream>
struct Access<__nv_bfloat16, 1, kStream> {
    static __device__ __forceinline__ void load(const __nv_bfloat16* p, float (&v)[1])
    {
        const unsigned short r = kStream ? __ldcs(reinterpret_cast<const unsigned short*>(p))
                                         : __ldg(reinterpret_cast<const unsigned short*>(p));
        v[0] = __uint_as_float(static_cast<uint32_t>(r) << 16);
    }
    static __device__ __forceinline__ void store(__nv_bfloat16* p, const float (&v)[1])
    {
        const __nv_bfloat16 r = __float2bfloat16_rn(v[0]);
        if (kStream) __stcs(reinterpret_cast<unsigned short*>(p),
                            *reinterpret_cast<const unsigned short*>(&r));
        else *p = r;
    }
};

}  // namespace affinescan
