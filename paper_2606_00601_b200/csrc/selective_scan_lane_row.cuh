// selective_scan_lane_row.cuh — variant AFFINESCAN_SELECTIVE_LANE_ROW of
// selective_scan_fwd (include/affinescan.h; BJ north_star).
//
// The many-rows schedule (cfg3).  G lanes share one (b,d) row (G = 1, 2 or 4); each lane keeps
// NS = 16/G of the row's N = 16 states h[n] and A2[n] = A[d,n]*log2(e) in registers, packed two
// states per 64-bit register pair, and walks L sequentially: no warp scan, no rescan.  Per pair
// of state-steps the work is
//     arg  = {delta,delta} * A2pair          FMUL2   (fma pipe, mul.rn.f32x2)
//     a    = 2^arg                           2 x MUFU.EX2   -- or, for a compile-time share of the
//                                            (timestep, pair) slots, a Cody-Waite + minimax
//                                            polynomial 2^x evaluated with FFMA2 on the fma pipe
//     u    = {delta*x,delta*x} * Bpair       FMUL2
//     h    = a*h + u                         FFMA2   (Eq.3 with the pair of P:86 Eq.6)
//     y   += Cpair*h                         FFMA2   (BJ: y = sum_n C h + D x; h never stored)
// issued "pass-major": one pass = four states over the VEC timesteps of a 128-bit group, first
// every 2^x of the pass, then the dependent h chains.
// A warp covers 32/G consecutive d of one batch b, so B_t/C_t are warp-uniform: each warp stages
// its [2][N][TC] B/C tile with two TMA tensor copies per tile (cp.async.bulk.tensor.2d through
// tensor maps over [batch*N, L], mbarrier complete_tx, double-buffered; SASS UTMALDG),
// transposes/widens it once to an fp32 [TC][2][N] tile, and every state-step then reads B/C with
// broadcast LDS.128.  x/delta come from global memory as raw 128-bit words prefetched two groups
// ahead; y is reduced across the G lanes of the row with a shuffle reduce-scatter and leaves
// with 128/G-bit stores.  Warps are autonomous: no CTA barrier.
//
// Template options:
//   EXT   the fused steps either side of the scan, a bit mask: kExtSoftplus =
//         Delta = softplus(delta + bias[d]); kExtGate = y <- y*silu(z); kExtReset = resets (the
//         pair of a reset step is the left zero (0, u_t)); kExtRuntime = each step is present only
//         if its pointer / flag in SelectiveExt says so (the generic instantiation).  The gated
//         Mamba block (softplus + bias + z, no resets) has its own branch-free instantiation.
//   ASTR  structured-A fast paths (P:118-122 generality): 0 = general A;
//         1 = one decay per row, A[d,n] = A[d,0] (one 2^x per (b,d,t));
//         2 = A[d,n] = (n+1) A[d,0]: a_n = r^(n+1), r = 2^(delta A2[d,0]) (one 2^x and a chain of
//             packed multiplies per (b,d,t)).
#pragma once

#include <type_traits>

#include "selective_common.cuh"
#include "tma.cuh"

namespace affinescan {

constexpr int kExtSoftplus = 1, kExtGate = 2, kExtReset = 4, kExtRuntime = 8;
constexpr int kExtGated = kExtSoftplus | kExtGate;                               // Mamba block
constexpr int kExtGeneric = kExtSoftplus | kExtGate | kExtReset | kExtRuntime;   // anything

// Which (timestep-in-group k, pair p) slots use the polynomial: F16 of every 16 slots, spread
// evenly (Bresenham), decided at compile time.
__host__ __device__ constexpr bool lane_row_slot_is_poly(int idx, int F16)
{
    return ((idx + 1) * F16) / 16 != (idx * F16) / 16;
}

// ------------------------------------------------------------------ shared-memory plan
template <typename T, int TC>
struct LaneRowSmem {
    static constexpr int N = 16;
    static constexpr int kRawPitch = TC * static_cast<int>(sizeof(T));  // bytes per box row
    static constexpr int kRawStage = 2 * N * kRawPitch;                 // B box then C box
    static constexpr int kBcTile = TC * 2 * N * 4;                      // fp32 [TC][2][N]
    static constexpr int kPerWarp = 2 * kRawStage + kBcTile + 128;      // + 2 mbarriers, padded
    static_assert(kRawStage % 256 == 0 && kPerWarp % 128 == 0, "TMA destinations: 128 B aligned");
};

// CNT consecutive io-dtype values at p <-> floats (16 / 8 / 4 / 2-byte accesses).
template <typename T, int CNT>
struct RowSeg;
template <>
struct RowSeg<float, 4> {
    static __device__ __forceinline__ void store(float* p, const float (&v)[4])
    {
        __stcs(reinterpret_cast<float4*>(p), make_float4(v[0], v[1], v[2], v[3]));
    }
    static __device__ __forceinline__ void load(const float* p, float (&v)[4])
    {
        const float4 r = __ldcs(reinterpret_cast<const float4*>(p));
        v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w;
    }
};
template <>
struct RowSeg<float, 2> {
    static __device__ __forceinline__ void store(float* p, const float (&v)[2])
    {
        __stcs(reinterpret_cast<float2*>(p), make_float2(v[0], v[1]));
    }
    static __device__ __forceinline__ void load(const float* p, float (&v)[2])
    {
        const float2 r = __ldcs(reinterpret_cast<const float2*>(p));
        v[0] = r.x; v[1] = r.y;
    }
};
template <>
struct RowSeg<float, 1> {
    static __device__ __forceinline__ void store(float* p, const float (&v)[1]) { __stcs(p, v[0]); }
    static __device__ __forceinline__ void load(const float* p, float (&v)[1]) { v[0] = __ldcs(p); }
};
template <>
struct RowSeg<__nv_bfloat16, 8> {
    static __device__ __forceinline__ void store(__nv_bfloat16* p, const float (&v)[8])
    {
        __stcs(reinterpret_cast<uint4*>(p),
               make_uint4(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3]),
                          pack_bf16x2(v[4], v[5]), pack_bf16x2(v[6], v[7])));
    }
    static __device__ __forceinline__ void load(const __nv_bfloat16* p, float (&v)[8])
    {
        unpack128<__nv_bfloat16>(__ldcs(reinterpret_cast<const uint4*>(p)), v);
    }
};
template <>
struct RowSeg<__nv_bfloat16, 4> {
    static __device__ __forceinline__ void store(__nv_bfloat16* p, const float (&v)[4])
    {
        __stcs(reinterpret_cast<uint2*>(p),
               make_uint2(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3])));
    }
    static __device__ __forceinline__ void load(const __nv_bfloat16* p, float (&v)[4])
    {
        const uint2 r = __ldcs(reinterpret_cast<const uint2*>(p));
        v[0] = bf16_lo(r.x); v[1] = bf16_hi(r.x); v[2] = bf16_lo(r.y); v[3] = bf16_hi(r.y);
    }
};
template <>
struct RowSeg<__nv_bfloat16, 2> {
    static __device__ __forceinline__ void store(__nv_bfloat16* p, const float (&v)[2])
    {
        __stcs(reinterpret_cast<unsigned*>(p), pack_bf16x2(v[0], v[1]));
    }
    static __device__ __forceinline__ void load(const __nv_bfloat16* p, float (&v)[2])
    {
        const unsigned r = __ldcs(reinterpret_cast<const unsigned*>(p));
        v[0] = bf16_lo(r); v[1] = bf16_hi(r);
    }
};

// ====================================================================================
// The kernel.  T = io dtype; G = lanes per row; TC = timesteps per staged B/C tile;
// WARPS = warps per CTA; F16 = sixteenths of the exponentials done by the polynomial;
// DEG = its degree; EXT / ASTR: see the header comment.
// ====================================================================================
template <typename T, int G, int TC, int WARPS, int F16, int DEG, int EXT, int ASTR>
__global__ void __launch_bounds__(WARPS * 32)
selective_scan_lane_row_kernel(const T* __restrict__ x, const T* __restrict__ delta,
                               const float* __restrict__ A,
                               const __grid_constant__ CUtensorMap mapB,
                               const __grid_constant__ CUtensorMap mapC,
                               const float* __restrict__ D,
                               const float* __restrict__ h0, T* __restrict__ y,
                               float* __restrict__ h_last, const SelectiveExt ext, int batch,
                               int d_inner, long long L)
{
    using S = LaneRowSmem<T, TC>;
    constexpr int N = S::N;
    constexpr int VEC = Io<T>::kVec;   // timesteps per 128-bit access
    constexpr int kChunks = TC / VEC;  // 128-bit chunks per raw row
    constexpr int RW = 32 / G;         // rows per warp
    constexpr int NS = N / G;          // states per lane
    constexpr int NP = NS / 2;         // packed pairs per lane
    constexpr int PP = 2;              // packed pairs per pass (four states share a MUFU burst)
    constexpr int YC = VEC / G;        // y values per lane after the reduce-scatter
    static_assert(G == 1 || G == 2 || G == 4, "G");
    static_assert(NP % PP == 0, "pairs per pass");
    static_assert(NS % 4 == 0 && YC >= 1 && TC % VEC == 0 && (TC / VEC) % 2 == 0, "shape");
    static_assert(ASTR == 0 || (G == 1 && F16 == 0), "structured-A paths: one lane per row, no polynomial");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int g = lane % G;  // which NS-slice of the row's states
    const long long rows = static_cast<long long>(batch) * d_inner;
    const long long row0 = (static_cast<long long>(blockIdx.x) * WARPS + warp) * RW;
    if (row0 >= rows) return;  // whole warp exits together; warps never sync with each other
    const long long row = row0 + lane / G;
    const int b = static_cast<int>(row0 / d_inner);  // d_inner % 32 == 0: uniform over the warp
    const int d = static_cast<int>(row - static_cast<long long>(b) * d_inner);

    unsigned char* wbase = smem_raw + static_cast<size_t>(warp) * S::kPerWarp;
    float* bc = reinterpret_cast<float*>(wbase + 2 * S::kRawStage);
    uint64_t* full = reinterpret_cast<uint64_t*>(wbase + 2 * S::kRawStage + S::kBcTile);

    if (lane == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        fence_mbar_init();
    }
    fence_proxy_async_smem();
    __syncwarp();

    const long long ntiles = (L + TC - 1) / TC;
    // A2 staging: one elected lane issues two tensor copies per tile: box {TC, N} of B[b] and
    // of C[b] (tensor maps over [batch*N, L]); the tail tile is zero-filled by the TMA unit.
    auto issue_tile = [&](long long tile) {
        if (lane == 0) {
            const int st = static_cast<int>(tile & 1);
            const int t0 = static_cast<int>(tile * TC);
            unsigned char* dst = wbase + st * S::kRawStage;
            mbar_arrive_expect_tx(&full[st], static_cast<unsigned>(S::kRawStage));
            tma_tile_2d_g2s(dst, &mapB, t0, b * N, &full[st]);
            tma_tile_2d_g2s(dst + N * S::kRawPitch, &mapC, t0, b * N, &full[st]);
        }
    };
    issue_tile(0);
    if (ntiles > 1) issue_tile(1);

    // per-row constants and state, packed two states per register pair
    pair_t A2p[NP], h2[NP];
    float amax = 0.0f;
#pragma unroll
    for (int q = 0; q < NS / 4; ++q) {
        const float4 av =
            __ldg(reinterpret_cast<const float4*>(A + static_cast<long long>(d) * N + g * NS) + q);
        A2p[2 * q + 0] = pk(av.x * kLog2e, av.y * kLog2e);
        A2p[2 * q + 1] = pk(av.z * kLog2e, av.w * kLog2e);
        amax = fmaxf(fmaxf(fabsf(av.x), fabsf(av.y)), fmaxf(fmaxf(fabsf(av.z), fabsf(av.w)), amax));
        float4 hv = make_float4(0.f, 0.f, 0.f, 0.f);
        if (h0) hv = __ldg(reinterpret_cast<const float4*>(h0 + row * N + g * NS) + q);
        h2[2 * q + 0] = pk(hv.x, hv.y);
        h2[2 * q + 1] = pk(hv.z, hv.w);
    }
    float A20 = 0.0f;  // structured-A paths read A[d,0] only
    if (ASTR != 0) A20 = __ldg(A + static_cast<long long>(d) * N) * kLog2e;
    // the polynomial is used only while |delta*A2| <= 126 for every state of the lane
    const float dmax = 126.0f / (amax * kLog2e);
    const float Dg = (D && g == 0) ? __ldg(D + d) : 0.0f;  // the skip term is added by one lane
    constexpr bool kRt = (EXT & kExtRuntime) != 0;
    const float bias = ((EXT & kExtSoftplus) && ext.delta_bias) ? __ldg(ext.delta_bias + d) : 0.0f;

    const T* xr = x + row * L;
    const T* dr = delta + row * L;
    T* yr = y + row * L;
    const T* zr = (EXT & kExtGate) ? static_cast<const T*>(ext.z) : nullptr;
    if ((EXT & kExtGate) && (!kRt || zr)) zr += row * L;
    const unsigned char* rst =
        ((EXT & kExtReset) && ext.reset) ? ext.reset + static_cast<long long>(b) * L : nullptr;
    // timestep offset, inside a VEC group, of the YC values this lane stores
    int yoff = 0;
    if (G >= 2) yoff += (g & (G / 2)) ? VEC / 2 : 0;
    if (G >= 4) yoff += (g & 1) ? VEC / 4 : 0;

    // A1: raw 128-bit prefetch, two groups (2*VEC timesteps) ahead
    constexpr int PD = 2;
    uint4 xq[PD], dq[PD];
#pragma unroll
    for (int i = 0; i < PD; ++i) {
        xq[i] = make_uint4(0, 0, 0, 0);
        dq[i] = make_uint4(0, 0, 0, 0);
        if (static_cast<long long>(i) * VEC < L) {
            xq[i] = __ldcs(reinterpret_cast<const uint4*>(xr) + i);
            dq[i] = __ldcs(reinterpret_cast<const uint4*>(dr) + i);
        }
    }

    for (long long tile = 0; tile < ntiles; ++tile) {
        const int st = static_cast<int>(tile & 1);
        const unsigned parity = static_cast<unsigned>((tile >> 1) & 1);
        const long long t0 = tile * TC;
        mbar_wait(&full[st], parity);
        __syncwarp();  // every lane is done reading the fp32 tile of the previous iteration
        // A2: widen + transpose raw [2N][TC] (io dtype) -> bc [TC][2][N] (fp32); the
        // transposed stores hit 32 distinct banks.
#pragma unroll
        for (int c = 0; c < kChunks; ++c) {
            float v[VEC];
            unpack128<T>(*reinterpret_cast<const uint4*>(wbase + st * S::kRawStage +
                                                         lane * S::kRawPitch + c * 16), v);
#pragma unroll
            for (int k = 0; k < VEC; ++k) bc[(c * VEC + k) * 2 * N + lane] = v[k];
        }
        __syncwarp();
        if (tile + 2 < ntiles) {
            fence_proxy_async_smem();  // generic reads of the raw stage before the async overwrite
            issue_tile(tile + 2);
        }

        // A3..A9: sequential in t
#pragma unroll 1
        for (int gi = 0; gi < kChunks; gi += PD) {
#pragma unroll
            for (int pi = 0; pi < PD; ++pi) {
                const int grp = gi + pi;
                const long long tg = t0 + grp * VEC;
                if (grp < kChunks && tg < L) {  // warp-uniform
                    float xv[VEC], dl[VEC];
                    unpack128<T>(xq[pi], xv);
                    unpack128<T>(dq[pi], dl);
                    if (tg + PD * VEC < L) {
                        xq[pi] = __ldcs(reinterpret_cast<const uint4*>(xr + tg + PD * VEC));
                        dq[pi] = __ldcs(reinterpret_cast<const uint4*>(dr + tg + PD * VEC));
                    }
                    // f1 prologue: Delta = softplus(delta + bias[d]); f2: reset bits of the group
                    unsigned rmask = 0;
                    float zv[YC];
                    if (EXT & kExtSoftplus) {
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            dl[k] += bias;
                            if (!kRt || ext.delta_softplus) dl[k] = softplus_f(dl[k]);
                        }
                    }
                    if ((EXT & kExtReset) && rst) {
#pragma unroll
                        for (int k = 0; k < VEC; ++k)
                            rmask |= (__ldg(rst + tg + k) != 0 ? 1u : 0u) << k;
                    }
                    if ((EXT & kExtGate) && (!kRt || zr)) RowSeg<T, YC>::load(zr + tg + yoff, zv);
                    float ys[VEC];
                    float dxs[VEC];
                    pair_t y2[VEC];
#pragma unroll
                    for (int k = 0; k < VEC; ++k) {
                        dxs[k] = dl[k] * xv[k];
                        y2[k] = pk(Dg * xv[k], 0.0f);
                    }
                    // structured A: the decay base r_k = 2^(delta_k A2[d,0]) of each timestep
                    pair_t cur[ASTR == 2 ? VEC : 1];
                    float r1[ASTR != 0 ? VEC : 1], r2[ASTR == 2 ? VEC : 1];
                    if (ASTR != 0) {
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            r1[k] = ex2_approx(dl[k] * A20);
                            if (ASTR == 2) {
                                r2[k] = r1[k] * r1[k];
                                cur[k] = pk(r1[k], r2[k]);  // {r^1, r^2}; next pairs: * {r^2, r^2}
                            }
                        }
                    }
                    // One pass = four states (two packed pairs, one LDS.128 of B and of C per
                    // timestep) over the VEC timesteps of the group: first every 2^x of the pass
                    // (independent: they stream through the MUFU / fma pipes back to back), then
                    // the two dependent h chains.  F = sixteenths of the exps taken by the
                    // polynomial (0 on the guarded slow path); RST = the group holds a reset.
                    auto pass = [&](int q, auto ftag, auto rtag) {
                        constexpr int F = decltype(ftag)::value;
                        constexpr bool RST = decltype(rtag)::value;
                        pair_t av[VEC][PP];
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            const pair_t dd = pk(dl[k], dl[k]);
#pragma unroll
                            for (int s = 0; s < PP; ++s) {
                                const int p = PP * q + s;
                                if (ASTR == 1) {
                                    av[k][s] = pk(r1[k], r1[k]);
                                } else if (ASTR == 2) {
                                    if (p > 0) cur[k] = mul2(cur[k], pk(r2[k], r2[k]));
                                    av[k][s] = cur[k];
                                } else if (lane_row_slot_is_poly(k * NP + p, F)) {
                                    av[k][s] = exp2_poly2<DEG>(dd, A2p[p]);
                                } else {
                                    float lo, hi;
                                    upk(mul2(dd, A2p[p]), lo, hi);
                                    av[k][s] = pk(ex2_approx(lo), ex2_approx(hi));
                                }
                                // a reset step is the left-zero pair (0, u_t): h_{t-1} is dropped
                                if (RST && ((rmask >> k) & 1u)) av[k][s] = pk(0.0f, 0.0f);
                            }
                        }
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            const pair_t dxx = pk(dxs[k], dxs[k]);
                            const float* bct = bc + (grp * VEC + k) * 2 * N + g * NS + 2 * PP * q;
#pragma unroll
                            for (int s = 0; s < PP; s += 2) {
                                const int p = PP * q + s;
                                const ulonglong2 b4 =
                                    *reinterpret_cast<const ulonglong2*>(bct + 2 * s);
                                const ulonglong2 c4 =
                                    *reinterpret_cast<const ulonglong2*>(bct + N + 2 * s);
                                h2[p] = fma2(av[k][s], h2[p], mul2(dxx, b4.x));
                                h2[p + 1] = fma2(av[k][s + 1], h2[p + 1], mul2(dxx, b4.y));
                                y2[k] = fma2(c4.x, h2[p], y2[k]);
                                y2[k] = fma2(c4.y, h2[p + 1], y2[k]);
                            }
                        }
                    };
                    // the polynomial needs |delta*A2| <= 126; a group in which any lane of the
                    // warp exceeds that (a underflows: far outside BJ's distributions) takes the
                    // all-MUFU path instead, so nothing is ever clamped
                    bool poly_ok = true;
                    if (F16 > 0) {
                        float dm = fabsf(dl[0]);
#pragma unroll
                        for (int k = 1; k < VEC; ++k) dm = fmaxf(dm, fabsf(dl[k]));
                        poly_ok = !__any_sync(kFullMask, !(dm <= dmax));
                    }
                    if ((EXT & kExtReset) && rmask != 0) {  // warp-uniform (rows of a warp share b)
#pragma unroll
                        for (int q = 0; q < NP / PP; ++q)
                            pass(q, std::integral_constant<int, 0>{}, std::true_type{});
                    } else if (poly_ok) {
#pragma unroll
                        for (int q = 0; q < NP / PP; ++q)
                            pass(q, std::integral_constant<int, F16>{}, std::false_type{});
                    } else {
#pragma unroll
                        for (int q = 0; q < NP / PP; ++q)
                            pass(q, std::integral_constant<int, 0>{}, std::false_type{});
                    }
#pragma unroll
                    for (int k = 0; k < VEC; ++k) {
                        float ylo, yhi;
                        upk(y2[k], ylo, yhi);
                        ys[k] = ylo + yhi;
                    }
                    // A9: reduce the partial sums over the G lanes of the row (reduce-scatter:
                    // each lane ends with YC fully reduced timesteps) and store
                    if (G >= 2) {
                        const bool up = (g & (G / 2)) != 0;
#pragma unroll
                        for (int j = 0; j < VEC / 2; ++j) {
                            const float mine = up ? ys[VEC / 2 + j] : ys[j];
                            const float send = up ? ys[j] : ys[VEC / 2 + j];
                            ys[j] = mine + __shfl_xor_sync(kFullMask, send, G / 2);
                        }
                    }
                    if (G >= 4) {
                        const bool up = (g & 1) != 0;
#pragma unroll
                        for (int j = 0; j < VEC / 4; ++j) {
                            const float mine = up ? ys[VEC / 4 + j] : ys[j];
                            const float send = up ? ys[j] : ys[VEC / 4 + j];
                            ys[j] = mine + __shfl_xor_sync(kFullMask, send, 1);
                        }
                    }
                    float out[YC];
#pragma unroll
                    for (int j = 0; j < YC; ++j) out[j] = ys[j];
                    if ((EXT & kExtGate) && (!kRt || zr)) {  // f1 epilogue: y <- y * silu(z)
#pragma unroll
                        for (int j = 0; j < YC; ++j) out[j] *= silu_io<T>(zv[j]);
                    }
                    if (y) RowSeg<T, YC>::store(yr + tg + yoff, out);  // y == NULL: aggregate-only call
                }
            }
        }
    }
    // A10: final state
    if (h_last) {
#pragma unroll
        for (int q = 0; q < NS / 4; ++q) {
            float a0, a1, a2, a3;
            upk(h2[2 * q + 0], a0, a1);
            upk(h2[2 * q + 1], a2, a3);
            reinterpret_cast<float4*>(h_last + row * N + g * NS)[q] = make_float4(a0, a1, a2, a3);
        }
    }
}

}  // namespace affinescan
