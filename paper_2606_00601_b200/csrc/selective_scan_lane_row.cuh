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
// issued "pass-major" for G = 1 (one pass = four states over the VEC timesteps of a 128-bit group,
// first every 2^x of the pass, then the dependent h chains) and timestep-major for G >= 2.
// A warp covers 32/G consecutive d of one batch b, so B_t/C_t are warp-uniform and are read from an
// fp32 [TC][2][N] shared-memory tile with broadcast LDS.128.  The tile is staged either by the warp
// itself (uniform grid: two TMA tensor copies per tile, cp.async.bulk.tensor.2d through tensor maps
// over [batch*N, L], mbarrier complete_tx, double-buffered, SASS UTMALDG; then widened/transposed by
// the warp) or once per CTA by a producer warp (balanced grid, selective_scan_lane_mix_kernel at
// the end of this file).  x/delta come from global memory as raw 128-bit words prefetched PD groups
// ahead; y is reduced across the G lanes of the row with a shuffle reduce-scatter and leaves with
// 128/G-bit stores.  Row warps never meet at a CTA barrier.
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

// compile-time loop: f(integral_constant<int, I>) for I in [0, N)
template <int I, int N, typename F>
__device__ __forceinline__ void static_for(F&& f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
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
// CTA-shared B/C tiles (lane_mix kernel): a producer warp stages the fp32 [TC][2][N] tiles of the
// batches the CTA touches into a ring of kStages slots; consumers wait on full[slot] and arrive
// on empty[slot] once per tile.
#ifndef LR_PD
#define LR_PD 2
#endif
#ifndef LR_MIX_STAGES
#define LR_MIX_STAGES 4
#endif
constexpr int kMixStages = LR_MIX_STAGES;
constexpr int kMixMaxBatches = 2;
struct SharedTiles {
    const float* bc;   // [kMixStages][kMixMaxBatches][TC][2][N]
    uint64_t* full;    // [kMixStages], count 1 (producer)
    uint64_t* empty;   // [kMixStages], count = consumer warps with work
    int bsel;          // which of the CTA's batches this warp's rows belong to
    // x / delta ring of the warp (XTMA): 2 stages x (x rows | delta rows), 128 B per row and stage
    // = kXGroups 128-bit groups, written by TMA tensor copies with the 128-byte swizzle
    unsigned char* xring;
    uint64_t* xfull;   // [2], count 1
    const CUtensorMap* mapX;
    const CUtensorMap* mapD;
};
constexpr int kXGroups = 8;              // 128-bit groups per row per ring stage
constexpr int kXPerWarp = 2 * 2 * 16 * 128;  // stages x arrays x rows (<= 16) x 128 B

// The staging duty of the balanced grid: TMA tensor copies of the raw [2N][TC] boxes of the CTA's
// batches into a two-slot raw ring, widened and transposed (lane j = raw row j) into the ring of
// fp32 tiles.  Run by ONE warp of the CTA — a row warp that stages tile i + kMixStages - 1 before
// it consumes tile i, or on its own when that warp has no rows.
template <typename T, int TC>
struct MixStager {
    using S = LaneRowSmem<T, TC>;
    const CUtensorMap* mapB;
    const CUtensorMap* mapC;
    float* bc_ring;
    unsigned char* raw_ring;
    uint64_t* full;
    uint64_t* empty;
    uint64_t* raw_full;
    int b_first, nb;
    long long ntiles;

    __device__ __forceinline__ void issue_raw(long long tile, int lane) const
    {
        if (lane == 0) {
            const int rs = static_cast<int>(tile & 1);
            const int t0 = static_cast<int>(tile * TC);
            mbar_arrive_expect_tx(&raw_full[rs], static_cast<unsigned>(nb * S::kRawStage));
            for (int j = 0; j < nb; ++j) {
                unsigned char* dst = raw_ring + (rs * kMixMaxBatches + j) * S::kRawStage;
                tma_tile_2d_g2s(dst, mapB, t0, (b_first + j) * S::N, &raw_full[rs]);
                tma_tile_2d_g2s(dst + S::N * S::kRawPitch, mapC, t0, (b_first + j) * S::N,
                                &raw_full[rs]);
            }
        }
    }
    __device__ __forceinline__ void stage(long long tile, int lane) const
    {
        constexpr int VEC = Io<T>::kVec;
        const int slot = static_cast<int>(tile % kMixStages);
        const int rs = static_cast<int>(tile & 1);
        if (tile >= kMixStages)  // every row warp is done with the tile that held this slot
            mbar_wait(&empty[slot], static_cast<unsigned>((tile / kMixStages - 1) & 1));
        mbar_wait(&raw_full[rs], static_cast<unsigned>((tile >> 1) & 1));
        for (int j = 0; j < nb; ++j) {
            const unsigned char* src =
                raw_ring + (rs * kMixMaxBatches + j) * S::kRawStage + lane * S::kRawPitch;
            float* dst = bc_ring + (slot * kMixMaxBatches + j) * (TC * 2 * S::N);
#pragma unroll
            for (int c = 0; c < TC / VEC; ++c) {
                float v[VEC];
                unpack128<T>(*reinterpret_cast<const uint4*>(src + c * 16), v);
#pragma unroll
                for (int k = 0; k < VEC; ++k) dst[(c * VEC + k) * 2 * S::N + lane] = v[k];
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&full[slot]);
        if (tile + 2 < ntiles) {
            fence_proxy_async_smem();  // generic reads of the raw slot before the async overwrite
            issue_raw(tile + 2, lane);
        }
    }
    // tiles 0 .. kMixStages - 2 (no slot is in use yet)
    __device__ __forceinline__ void prologue(int lane) const
    {
        issue_raw(0, lane);
        if (ntiles > 1) issue_raw(1, lane);
        for (long long t = 0; t < kMixStages - 1 && t < ntiles; ++t) stage(t, lane);
    }
};

// The work of ONE warp: RW = 32/G consecutive rows starting at row0 (all in one batch), walked
// over the whole of L.  SHARED == false: `wbase` is the warp's private
// LaneRowSmem<T, TC>::kPerWarp bytes and the warp stages its own B/C tiles; SHARED == true: the
// tiles come from `sh`.
template <typename T, int G, int TC, int F16, int DEG, int EXT, int ASTR, int ORDER,
          bool SHARED = false, bool XTMA = false>
__device__ __forceinline__ void
lane_row_warp(const T* __restrict__ x, const T* __restrict__ delta, const float* __restrict__ A,
              const CUtensorMap* mapB, const CUtensorMap* mapC, const float* __restrict__ D,
              const float* __restrict__ h0, T* __restrict__ y, float* __restrict__ h_last,
              const SelectiveExt& ext, int d_inner, long long L, long long row0,
              unsigned char* wbase, const SharedTiles sh = SharedTiles{},
              const MixStager<T, TC>* stg = nullptr)
{
    using S = LaneRowSmem<T, TC>;
    constexpr int N = S::N;
    constexpr int VEC = Io<T>::kVec;   // timesteps per 128-bit access
    constexpr int kChunks = TC / VEC;  // 128-bit chunks per raw row
    constexpr int NS = N / G;          // states per lane
    constexpr int NP = NS / 2;         // packed pairs per lane
    constexpr int PP = 2;              // packed pairs per pass (four states share a MUFU burst)
    constexpr int YC = VEC / G;        // y values per lane after the reduce-scatter
    static_assert(G == 1 || G == 2 || G == 4, "G");
    static_assert(NP % PP == 0, "pairs per pass");
    static_assert(NS % 4 == 0 && YC >= 1 && TC % VEC == 0 && (TC / VEC) % LR_PD == 0, "shape");
    static_assert(ASTR == 0 || (G == 1 && F16 == 0), "structured-A paths: one lane per row, no polynomial");

    const int lane = threadIdx.x & 31;
    const int g = lane % G;  // which NS-slice of the row's states
    const long long row = row0 + lane / G;
    const int b = static_cast<int>(row0 / d_inner);  // d_inner % (32/G) == 0: uniform over the warp
    const int d = static_cast<int>(row - static_cast<long long>(b) * d_inner);

    const float* bc = SHARED ? sh.bc : reinterpret_cast<const float*>(wbase + 2 * S::kRawStage);
    float* bcw = SHARED ? nullptr : reinterpret_cast<float*>(wbase + 2 * S::kRawStage);
    uint64_t* full =
        SHARED ? sh.full : reinterpret_cast<uint64_t*>(wbase + 2 * S::kRawStage + S::kBcTile);

    if (!SHARED) {
        if (lane == 0) {
            mbar_init(&full[0], 1);
            mbar_init(&full[1], 1);
            fence_mbar_init();
        }
        fence_proxy_async_smem();
        __syncwarp();
    }

    const long long ntiles = (L + TC - 1) / TC;
    // A2 staging: one elected lane issues two tensor copies per tile: box {TC, N} of B[b] and
    // of C[b] (tensor maps over [batch*N, L]); the tail tile is zero-filled by the TMA unit.
    auto issue_tile = [&](long long tile) {
        if (!SHARED && lane == 0) {
            const int st = static_cast<int>(tile & 1);
            const int t0 = static_cast<int>(tile * TC);
            unsigned char* dst = wbase + st * S::kRawStage;
            mbar_arrive_expect_tx(&full[st], static_cast<unsigned>(S::kRawStage));
            tma_tile_2d_g2s(dst, mapB, t0, b * N, &full[st]);
            tma_tile_2d_g2s(dst + N * S::kRawPitch, mapC, t0, b * N, &full[st]);
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

    // A1 (XTMA): the warp's rows of x and delta come through its own shared-memory ring, one
    // 128-byte row segment (kXGroups groups) per row and stage, filled by TMA tensor copies of
    // boxes {128 B, 8 rows} with the 128-byte swizzle: the strided per-row global loads (one L1
    // wavefront per row and instruction) become two conflict-free LDS.128 per group.
    static_assert(!XTMA || (SHARED && G >= 2 && kXGroups % (TC / VEC) == 0), "x ring");
    constexpr int kXRows = 32 / G;
    constexpr int kXArray = kXRows * 128;
    constexpr int kXStage = 2 * kXArray;
    const long long nxblocks = (L + kXGroups * VEC - 1) / (kXGroups * VEC);
    auto issue_x = [&](long long blk) {
        if (XTMA && lane == 0) {
            const int xs = static_cast<int>(blk & 1);
            const int t0 = static_cast<int>(blk * (kXGroups * VEC));
            unsigned char* dst = sh.xring + xs * kXStage;
            mbar_arrive_expect_tx(&sh.xfull[xs], static_cast<unsigned>(kXStage));
#pragma unroll
            for (int bx = 0; bx < kXRows / 8; ++bx) {
                tma_tile_2d_g2s(dst + bx * 1024, sh.mapX, t0, static_cast<int>(row0) + bx * 8,
                                &sh.xfull[xs]);
                tma_tile_2d_g2s(dst + kXArray + bx * 1024, sh.mapD, t0,
                                static_cast<int>(row0) + bx * 8, &sh.xfull[xs]);
            }
        }
    };
    if (XTMA) {  // (the CTA initialised sh.xfull[0..1], count 1)
        issue_x(0);
        if (nxblocks > 1) issue_x(1);
    }
    // this lane's row inside the ring: box (row / 8), line (row % 8), chunks XOR-swizzled by line
    const int xline = (lane / G) & 7;
    const int xrowoff = ((lane / G) >> 3) * 1024 + xline * 128;

    // A1 (no XTMA): raw 128-bit prefetch, PD groups (PD*VEC timesteps) ahead
    constexpr int PD = LR_PD;  // 128-bit x/delta groups in flight per row
    uint4 xq[PD], dq[PD];
#pragma unroll
    for (int i = 0; i < PD; ++i) {
        xq[i] = make_uint4(0, 0, 0, 0);
        dq[i] = make_uint4(0, 0, 0, 0);
        if (!XTMA && static_cast<long long>(i) * VEC < L) {
            xq[i] = __ldcs(reinterpret_cast<const uint4*>(xr) + i);
            dq[i] = __ldcs(reinterpret_cast<const uint4*>(dr) + i);
        }
    }

    if (XTMA) {  // words of group 0 (chunk 0 of block 0: swizzled position = xline)
        mbar_wait(&sh.xfull[0], 0u);
        const unsigned char* p0 = sh.xring + xrowoff + (xline << 4);
        xq[0] = lds128(p0);
        dq[0] = lds128(p0 + kXArray);
    }
    if (SHARED && stg) stg->prologue(lane);
    for (long long tile = 0; tile < ntiles; ++tile) {
        const long long t0 = tile * TC;
        int slot = 0;
        if (SHARED) {
            if (stg && tile + kMixStages - 1 < ntiles) stg->stage(tile + kMixStages - 1, lane);
            slot = static_cast<int>(tile % kMixStages);
            mbar_wait(&full[slot], static_cast<unsigned>((tile / kMixStages) & 1));
            bc = sh.bc + (slot * kMixMaxBatches + sh.bsel) * (TC * 2 * N);
        } else {
            const int st = static_cast<int>(tile & 1);
            const unsigned parity = static_cast<unsigned>((tile >> 1) & 1);
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
                for (int k = 0; k < VEC; ++k) bcw[(c * VEC + k) * 2 * N + lane] = v[k];
            }
            __syncwarp();
            if (tile + 2 < ntiles) {
                fence_proxy_async_smem();  // generic reads of the raw stage before the async overwrite
                issue_tile(tile + 2);
            }
        }

        // A3..A9: sequential in t.  One group = VEC timesteps of the warp's rows.
        // x ring: the tile lies inside one ring block
        const long long xblk = (tile * kChunks) / kXGroups;
        const int xcb = static_cast<int>((tile * kChunks) % kXGroups);
        const int xs = static_cast<int>(xblk & 1);
        const unsigned char* xbase = XTMA ? sh.xring + xs * kXStage + xrowoff : nullptr;

        // `fasttag`: the group and its prefetch refill lie inside the row, so every address is the
        // tile's base pointer plus a constant (no 64-bit position arithmetic per group)
        auto group = [&](auto pitag, auto fasttag, const int grp, const long long tg, const T* xg,
                         const T* dg, T* yg) {
            constexpr int PI = decltype(pitag)::value;
            constexpr bool FAST = decltype(fasttag)::value;
            float xv[VEC], dl[VEC];
            if (XTMA) {
                // this group's words were read from the ring one group ago; now read the next
                // group's (the first group of the next block waits for that block's copies)
                unpack128<T>(xq[0], xv);
                unpack128<T>(dq[0], dl);
                const int c1 = xcb + grp + 1;
                if (c1 < kXGroups) {
                    const int chunk = (c1 ^ xline) << 4;
                    xq[0] = lds128(xbase + chunk);
                    dq[0] = lds128(xbase + kXArray + chunk);
                } else {
                    if (xblk + 1 < nxblocks) {
                        mbar_wait(&sh.xfull[xs ^ 1], static_cast<unsigned>(((xblk + 1) >> 1) & 1));
                        const unsigned char* nb = sh.xring + (xs ^ 1) * kXStage + xrowoff + (xline << 4);
                        xq[0] = lds128(nb);
                        dq[0] = lds128(nb + kXArray);
                    }
                    // every word of this block is in registers: refill its stage
                    __syncwarp();
                    if (xblk + 2 < nxblocks) {
                        fence_proxy_async_smem();
                        issue_x(xblk + 2);
                    }
                }
            } else {
                unpack128<T>(xq[PI], xv);
                unpack128<T>(dq[PI], dl);
            }
            if (!XTMA) {   // refill the prefetch slot.  G >= 2 (four warps per sub-partition): always,
                // past the end of the row this group is re-read and never used (a
                // conditional refill costs a register copy per word: +2.5 %); G = 1:
                // conditional (measured: the unconditional form is scheduled late and
                // the one or two resident warps cannot hide it: 0.355 -> 0.425 ms)
                if (FAST) {
                    xq[PI] = __ldcs(reinterpret_cast<const uint4*>(xg + PD * VEC));
                    dq[PI] = __ldcs(reinterpret_cast<const uint4*>(dg + PD * VEC));
                } else {
                    const long long tn = tg + PD * VEC;
                    const long long ta = (G >= 2 && tn >= L) ? tg : tn;
                    if (G >= 2 || tn < L) {
                        xq[PI] = __ldcs(reinterpret_cast<const uint4*>(xr + ta));
                        dq[PI] = __ldcs(reinterpret_cast<const uint4*>(dr + ta));
                    }
                }
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
                            lds128_u64x2(bct + 2 * s);
                        const ulonglong2 c4 =
                            lds128_u64x2(bct + N + 2 * s);
                        h2[p] = fma2(av[k][s], h2[p], mul2(dxx, b4.x));
                        h2[p + 1] = fma2(av[k][s + 1], h2[p + 1], mul2(dxx, b4.y));
                        y2[k] = fma2(c4.x, h2[p], y2[k]);
                        y2[k] = fma2(c4.y, h2[p + 1], y2[k]);
                    }
                }
            };
            // ORDER == 1: timestep-major.  All the states of a lane for one timestep, then
            // the next timestep: the MUFU, fma-pipe and LDS instructions of a warp come
            // evenly mixed instead of in bursts (a burst of 2^x fills the SMSP's shared
            // MIO queue and stalls the other warps' LDS: measured with 4 warps per SMSP).
            auto steps = [&](auto ftag, auto rtag) {
                constexpr int F = decltype(ftag)::value;
                constexpr bool RST = decltype(rtag)::value;
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    const pair_t dd = pk(dl[k], dl[k]);
                    const pair_t dxx = pk(dxs[k], dxs[k]);
                    const float* bct = bc + (grp * VEC + k) * 2 * N + g * NS;
                    const bool rs = RST && ((rmask >> k) & 1u);
#pragma unroll
                    for (int p = 0; p < NP; p += 2) {
                        const ulonglong2 b4 = lds128_u64x2(bct + 2 * p);
                        const ulonglong2 c4 =
                            lds128_u64x2(bct + N + 2 * p);
                        pair_t a2[2];
#pragma unroll
                        for (int s = 0; s < 2; ++s) {
                            if (ASTR == 1) {
                                a2[s] = pk(r1[k], r1[k]);
                            } else if (ASTR == 2) {
                                if (p + s > 0) cur[k] = mul2(cur[k], pk(r2[k], r2[k]));
                                a2[s] = cur[k];
                            } else if (lane_row_slot_is_poly(k * NP + p + s, F)) {
                                a2[s] = exp2_poly2<DEG>(dd, A2p[p + s]);
                            } else {
                                float lo, hi;
                                upk(mul2(dd, A2p[p + s]), lo, hi);
                                a2[s] = pk(ex2_approx(lo), ex2_approx(hi));
                            }
                            if (rs) a2[s] = pk(0.0f, 0.0f);
                        }
                        h2[p] = fma2(a2[0], h2[p], mul2(dxx, b4.x));
                        h2[p + 1] = fma2(a2[1], h2[p + 1], mul2(dxx, b4.y));
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
            if (ORDER == 1) {
                if ((EXT & kExtReset) && rmask != 0)
                    steps(std::integral_constant<int, 0>{}, std::true_type{});
                else if (poly_ok) steps(std::integral_constant<int, F16>{}, std::false_type{});
                else steps(std::integral_constant<int, 0>{}, std::false_type{});
            } else if ((EXT & kExtReset) && rmask != 0) {  // warp-uniform (rows of a warp share b)
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
            if (y) RowSeg<T, YC>::store(yg, out);  // y == NULL: aggregate-only call
        };
        if (G >= 2 && t0 + TC + PD * VEC <= L) {  // tile and its prefetch inside the row
            const T* xp = xr + t0;
            const T* dp = dr + t0;
            T* yp = yr + t0 + yoff;
#pragma unroll 1
            for (int gi = 0; gi < kChunks; gi += PD) {
                static_for<0, PD>([&](auto pi) {
                    constexpr int PI = decltype(pi)::value;
                    group(pi, std::true_type{}, gi + PI, t0 + (gi + PI) * VEC, xp + PI * VEC,
                          dp + PI * VEC, yp + PI * VEC);
                });
                xp += PD * VEC;
                dp += PD * VEC;
                yp += PD * VEC;
            }
        } else {
#pragma unroll 1
            for (int gi = 0; gi < kChunks; gi += PD)
                static_for<0, PD>([&](auto pi) {
                    constexpr int PI = decltype(pi)::value;
                    const long long tg = t0 + (gi + PI) * VEC;
                    if (tg < L) group(pi, std::false_type{}, gi + PI, tg, xr + tg, dr + tg, yr + tg + yoff);
                });
        }
        if (SHARED) {  // this warp is done with the slot
            __syncwarp();
            if (lane == 0) mbar_arrive(&sh.empty[slot]);
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

// ====================================================================================
// Uniform grid: every warp of every CTA takes the next 32/G rows.
// ====================================================================================
template <typename T, int G, int TC, int WARPS, int F16, int DEG, int EXT, int ASTR, int ORDER = 0>
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
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5;
    const long long rows = static_cast<long long>(batch) * d_inner;
    const long long row0 = (static_cast<long long>(blockIdx.x) * WARPS + warp) * (32 / G);
    if (row0 >= rows) return;  // whole warp exits together; warps never sync with each other
    lane_row_warp<T, G, TC, F16, DEG, EXT, ASTR, ORDER>(
        x, delta, A, &mapB, &mapC, D, h0, y, h_last, ext, d_inner, L, row0,
        smem_raw + static_cast<size_t>(warp) * LaneRowSmem<T, TC>::kPerWarp);
}

// ====================================================================================
// Balanced grid (one CTA of 16 row warps per SM): the XU pipe of a sub-partition
// is the wall, and with R rows the uniform grid leaves sub-partitions holding ceil(...) warps
// next to ones holding floor(...).  Here every sub-partition gets q2 G = 2 warps (16 rows each)
// and q4 G = 4 warps (8 rows), chosen by the host from the row count; for cfg3 three and one:
// 56 rows = 7/8 of what two G = 1 warps carry, spread over four warps whose MUFU, fma and LDS
// instructions interleave.  Warp w of a CTA runs on sub-partition w % 4.  CTA c owns rows
// [R c, R c + R) of a round, R = 64 q2 + 32 q4 (rounds of grid * R rows): the first 64 q2 go to
// the G = 2 warps, the rest to the G = 4 warps.  Those rows lie in
// at most kMixMaxBatches batches (the launcher checks d_inner), whose B/C tiles one of the
// G = 4 warps (MixStager) stages ONCE for the whole CTA, kMixStages - 1 tiles ahead of its own row work: TMA tensor copies of the raw [2N][TC] boxes into a
// two-slot raw ring, widened and transposed into a kMixStages-deep ring of fp32 [TC][2][N]
// tiles that the row warps read with broadcast LDS.128.
// ====================================================================================
template <typename T, int TC>
struct LaneMixSmem {
    using S = LaneRowSmem<T, TC>;
    static constexpr int kXBytes = 16 * kXPerWarp;  // x/delta rings of the 16 row warps (first:
                                                    // the swizzled boxes want 1024-byte alignment)
    static constexpr int kBcBytes = kMixStages * kMixMaxBatches * S::kBcTile;
    static constexpr int kRawBytes = 2 * kMixMaxBatches * S::kRawStage;
    static constexpr int kBarOffset = kXBytes + kBcBytes + kRawBytes;
    // full[], empty[], raw_full[2], xfull[16][2]; + 1024 to align the base
    static constexpr int kBytes = kBarOffset + (2 * kMixStages + 2 + 32) * 8 + 64 + 1024;
};

template <typename T, int TC, int F16, int DEG, int EXT, int ORDER>
__global__ void __launch_bounds__(16 * 32, 1)
selective_scan_lane_mix_kernel(const T* __restrict__ x, const T* __restrict__ delta,
                               const float* __restrict__ A,
                               const __grid_constant__ CUtensorMap mapB,
                               const __grid_constant__ CUtensorMap mapC,
                               const __grid_constant__ CUtensorMap mapX,
                               const __grid_constant__ CUtensorMap mapD,
                               const float* __restrict__ D,
                               const float* __restrict__ h0, T* __restrict__ y,
                               float* __restrict__ h_last, const SelectiveExt ext, int batch,
                               int d_inner, long long L, int q2, int q4)
{
    using M = LaneMixSmem<T, TC>;
    // composition of every sub-partition: q2 G = 2 warps (16 rows) and q4 G = 4 warps (8 rows),
    // q2 + q4 <= 4; warp w = slot * 4 + sub-partition.  The CTA's rows: 64 q2 for the G = 2 warps,
    // then 32 q4 for the G = 4 warps.
    const int kRowsPerCta = 64 * q2 + 32 * q4;
    // the last slot's warp on sub-partition 0 also stages the CTA's B/C tiles
    const int kStagerWarp = (q2 + q4 - 1) * 4;
    // x / delta through the per-warp TMA ring: plain form only (measured: the fused forms, which
    // also stream z, lose 6 % with it; the plain form gains 1 % and frees 12 % of the L1 data pipe)
    constexpr bool kXtma = EXT == 0;
    extern __shared__ __align__(128) unsigned char smem_dyn[];
    unsigned char* smem_raw = reinterpret_cast<unsigned char*>(
        (reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~static_cast<uintptr_t>(1023));
    float* bc_ring = reinterpret_cast<float*>(smem_raw + M::kXBytes);
    unsigned char* raw_ring = smem_raw + M::kXBytes + M::kBcBytes;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + M::kBarOffset);
    uint64_t* empty = full + kMixStages;
    uint64_t* raw_full = empty + kMixStages;
    uint64_t* xfull = raw_full + 2;  // [16 warps][2]

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const long long rows = static_cast<long long>(batch) * d_inner;
    const long long per_round = static_cast<long long>(gridDim.x) * kRowsPerCta;
    const long long ntiles = (L + TC - 1) / TC;

    for (long long base = 0; base < rows; base += per_round) {
        const long long cta0 = base + static_cast<long long>(blockIdx.x) * kRowsPerCta;
        if (cta0 >= rows) break;  // CTA-uniform
        const long long cta_rows = rows - cta0 < kRowsPerCta ? rows - cta0 : kRowsPerCta;
        // rows of this CTA: G = 2 warps take 16 each from the front, G = 4 warps 8 each after them
        // (cta_rows % 32 == 0)
        const long long r2 = cta_rows < 64 * q2 ? cta_rows : 64 * q2;
        const int n2 = static_cast<int>(r2 / 16);
        const int n4 = static_cast<int>((cta_rows - r2) / 8);
        const int b_first = static_cast<int>(cta0 / d_inner);
        const int nb = static_cast<int>((cta0 + cta_rows - 1) / d_inner) - b_first + 1;
        __syncthreads();  // previous round's barriers are quiet
        if (threadIdx.x == 0) {
            // a used mbarrier must be invalidated before it is initialised again
            if (base != 0) {
                for (int s = 0; s < 2 * kMixStages + 2 + 32; ++s) mbar_inval(&full[s]);
            }
#pragma unroll
            for (int s = 0; s < kMixStages; ++s) {
                mbar_init(&full[s], 1);
                mbar_init(&empty[s], n2 + n4);
            }
            mbar_init(&raw_full[0], 1);
            mbar_init(&raw_full[1], 1);
            for (int s = 0; s < 32; ++s) mbar_init(&xfull[s], 1);  // x rings: [warp][2]
            fence_mbar_init();
        }
        fence_proxy_async_smem();
        __syncthreads();

        MixStager<T, TC> stager;
        stager.mapB = &mapB;
        stager.mapC = &mapC;
        stager.bc_ring = bc_ring;
        stager.raw_ring = raw_ring;
        stager.full = full;
        stager.empty = empty;
        stager.raw_full = raw_full;
        stager.b_first = b_first;
        stager.nb = nb;
        stager.ntiles = ntiles;
        SharedTiles sh;
        sh.bc = bc_ring;
        sh.full = full;
        sh.empty = empty;
        sh.bsel = 0;
        sh.xring = smem_raw + warp * kXPerWarp;
        sh.xfull = xfull + 2 * warp;
        sh.mapX = &mapX;
        sh.mapD = &mapD;
        const int slot = warp >> 2, sp = warp & 3;
        const MixStager<T, TC>* stg = warp == kStagerWarp ? &stager : nullptr;
        bool worked = false;
        if (slot < q2) {
            const int i2 = slot * 4 + sp;
            if (i2 < n2) {
                const long long row0 = cta0 + i2 * 16;
                sh.bsel = static_cast<int>(row0 / d_inner) - b_first;
                lane_row_warp<T, 2, TC, F16, DEG, EXT, 0, ORDER, true, kXtma>(
                    x, delta, A, &mapB, &mapC, D, h0, y, h_last, ext, d_inner, L, row0, nullptr, sh,
                    stg);
                worked = true;
            }
        } else if (slot < q2 + q4) {
            const int i4 = (slot - q2) * 4 + sp;
            if (i4 < n4) {
                const long long row0 = cta0 + r2 + i4 * 8;
                sh.bsel = static_cast<int>(row0 / d_inner) - b_first;
                lane_row_warp<T, 4, TC, F16, DEG, EXT, 0, ORDER, true, kXtma>(
                    x, delta, A, &mapB, &mapC, D, h0, y, h_last, ext, d_inner, L, row0, nullptr, sh,
                    stg);
                worked = true;
            }
        }
        if (stg && !worked) {
            // a last CTA without rows for this warp: staging only
            stager.issue_raw(0, lane);
            if (ntiles > 1) stager.issue_raw(1, lane);
            for (long long tile = 0; tile < ntiles; ++tile) stager.stage(tile, lane);
        }
    }
}

}  // namespace affinescan
