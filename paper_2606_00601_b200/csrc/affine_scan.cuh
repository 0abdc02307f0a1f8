// affine_scan.cuh — kernels for affine_scan (include/affinescan.h):
//   h[s,t] = a[s,t]*h[s,t-1] + u[s,t]   as a prefix scan over pairs (a_t,u_t) under
//   (A2,U2)(+)(A1,U1) = (A2*A1, A2*U1+U2)           (Eq.6, Eq.7)
//
// Schedule (BJ north_star; SURVEY §8a A1,A4-A8,A11): coalesced 128-bit loads; every
// thread composes its VEC consecutive steps in registers; pairs are combined across
// the warp with __shfl_up_sync and across warps through shared memory; the carry
// crosses tiles either by decoupled look-back over a flattened [num_seq*L] stream
// (sequence heads become reset pairs (0, a0*h0+u0), a left zero of (+)) or in a
// CTA loop with the carry in a register.  The paper's Blelloch up/down-sweep
// is kept as a shared-memory ablation only.
#pragma once

#include "common.cuh"
#include "tma.cuh"

namespace affinescan {

// ------------------------------------------------------------------ tile descriptors
// One descriptor per tile = two 64-bit words {status:32 | float bits:32}: word 0 carries
// P, word 1 carries U.  Each word is written with ONE 64-bit store, so a reader that
// sees equal valid statuses in both words holds a consistent pair.  INCLUSIVE
// descriptors carry (0, h_end): the state after the tile, as a left-zero pair.
// status = (tag << 2) | state with tag = the launch's epoch + 1 (never 0): words left by an
// earlier launch, or the zero fill of a fresh buffer, read as EMPTY, so the descriptors are
// never cleared between calls.  The control block holds the tile ticket, the count of finished
// tiles and the epoch; the last tile to finish resets the first two and bumps the epoch, which
// also makes a captured CUDA graph replayable.
constexpr unsigned kDescEmpty = 0u;
constexpr unsigned kDescAggregate = 1u;
constexpr unsigned kDescInclusive = 2u;

struct LookbackCtrl {
    unsigned ticket;
    unsigned done;
    unsigned epoch;
    unsigned pad;
};

__device__ __forceinline__ void desc_store(unsigned long long* d, unsigned tag, unsigned state,
                                           Pair v)
{
    const unsigned long long hi = static_cast<unsigned long long>((tag << 2) | state) << 32;
    const unsigned long long w0 = hi | __float_as_uint(v.P);
    const unsigned long long w1 = hi | __float_as_uint(v.U);
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(d), "l"(w0) : "memory");
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(d + 1), "l"(w1) : "memory");
}

__device__ __forceinline__ unsigned desc_load(const unsigned long long* d, unsigned tag, Pair& v)
{
    unsigned long long w0, w1;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(w0) : "l"(d) : "memory");
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(w1) : "l"(d + 1) : "memory");
    const unsigned s0 = static_cast<unsigned>(w0 >> 32);
    const unsigned s1 = static_cast<unsigned>(w1 >> 32);
    v.P = __uint_as_float(static_cast<unsigned>(w0));
    v.U = __uint_as_float(static_cast<unsigned>(w1));
    // another epoch's word, or a torn read (mid-transition) => EMPTY: retry
    return (s0 == s1 && (s0 >> 2) == (tag & 0x3fffffffu)) ? (s0 & 3u) : kDescEmpty;
}

// ------------------------------------------------------------------ per-thread tile state
// A CTA tile is WARPS*32*VEC*J elements.  Warp w owns a contiguous 32*VEC*J slice; inside
// it, lane l's j-th vector starts at j*32*VEC + l*VEC, so every 128-bit access of a warp
// is one fully coalesced 512-byte request.
template <int VEC, int J>
struct TileRegs {
    float av[J][VEC];
    float uv[J][VEC];
    Pair excl[J];  // composition of lanes < lane within vector-row j
    Pair tot[J];   // composition of all 32 lanes of vector-row j
};

// Thread-local compose + warp combine (A5) of one vector-row.
template <int VEC, int J>
__device__ __forceinline__ void row_scan(TileRegs<VEC, J>& r, int j, int lane)
{
    Pair loc{r.av[j][0], r.uv[j][0]};
#pragma unroll
    for (int k = 1; k < VEC; ++k) loc = compose(Pair{r.av[j][k], r.uv[j][k]}, loc);
    const Pair inc = warp_inclusive_scan(loc, lane);
    Pair ex = shfl_up_pair(inc, 1);
    if (lane == 0) ex = identity_pair();
    r.excl[j] = ex;
    r.tot[j] = shfl_pair(inc, 31);
}

template <int VEC, int J>
__device__ __forceinline__ Pair warp_total(const TileRegs<VEC, J>& r)
{
    Pair w = r.tot[0];
#pragma unroll
    for (int j = 1; j < J; ++j) w = compose(r.tot[j], w);
    return w;
}

// Position of flat element index base+off inside its sequence: (s, t).  q0 = base / L and
// r0 = base % L are computed once per tile; off < tile size < 2^31.
__device__ __forceinline__ void seq_pos(long long q0, long long r0, int off, long long L,
                                        int tile_elems, long long& s, long long& t)
{
    t = r0 + off;
    s = q0;
    if (t >= L) {
        if (L >= tile_elems) {  // at most one sequence boundary inside the tile
            t -= L;
            s += 1;
        } else {  // t < L + tile_elems < 2^32
            const unsigned q = static_cast<unsigned>(t) / static_cast<unsigned>(L);
            t -= static_cast<long long>(q) * L;
            s += q;
        }
    }
}

// ------------------------------------------------------------------ decoupled look-back
// Run by one warp.  Publishes the tile's descriptor (AGGREGATE, or INCLUSIVE at once when the
// tile needs no carry-in: it starts at a sequence head, or its product is exactly 0), walks the
// predecessors 32 at a time until an INCLUSIVE one, publishes INCLUSIVE, and returns the state
// entering the tile.
__device__ __forceinline__ float lookback_carry(unsigned long long* __restrict__ desc,
                                                unsigned tile, unsigned tag, Pair agg,
                                                bool need_carry, int lane)
{
    unsigned long long* my = desc + 2ull * tile;
    const bool self_contained = (agg.P == 0.0f) || !need_carry;
    if (lane == 0) {
        if (self_contained) desc_store(my, tag, kDescInclusive, Pair{0.0f, agg.U});
        else desc_store(my, tag, kDescAggregate, agg);
    }
    float h_in = 0.0f;
    if (need_carry) {
        Pair acc = identity_pair();  // (+) of the tiles examined so far (later side)
        long long look = static_cast<long long>(tile) - 1;
        while (true) {
            const long long idx = look - lane;
            Pair e{0.0f, 0.0f};
            unsigned st = kDescInclusive;  // before the stream: state 0
            if (idx >= 0) {
                const unsigned long long* d = desc + 2ull * idx;
                st = desc_load(d, tag, e);
                while (st == kDescEmpty) {  // back off: the poll competes with the data stream
                    __nanosleep(64);
                    st = desc_load(d, tag, e);
                }
            }
            __syncwarp();
            const unsigned incl = __ballot_sync(kFullMask, st == kDescInclusive);
            const int first = incl ? (__ffs(incl) - 1) : 32;
            if (lane > first) e = identity_pair();
            // ordered tree reduction: lane 0 holds the LATEST tile (left operand)
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const Pair o = shfl_down_pair(e, d);
                if (lane + d < 32) e = compose(e, o);
            }
            const Pair win = shfl_pair(e, 0);
            acc = compose(acc, win);
            if (incl) break;
            look -= 32;
        }
        h_in = acc.U;  // acc.P == 0: the chain ended at an inclusive (left-zero) pair
        if (lane == 0 && !self_contained)
            desc_store(my, tag, kDescInclusive, Pair{0.0f, apply(agg, h_in)});
    }
    return h_in;
}

// ====================================================================================
// Variant AFFINESCAN_AFFINE_LOOKBACK: single pass, decoupled look-back
// ====================================================================================
template <typename T, int VEC, int J, int WARPS>
// 4 CTAs / SM (<= 64 registers): tiles in their load phase cover the ones that look back
__global__ void __launch_bounds__(WARPS * 32, 1024 / (WARPS * 32))
affine_scan_lookback_kernel(const T* __restrict__ a, const T* __restrict__ u,
                            const float* __restrict__ h0, T* __restrict__ h,
                            float* __restrict__ h_last, long long total, long long L,
                            unsigned long long* __restrict__ desc, LookbackCtrl* __restrict__ ctrl)
{
    constexpr int kWarpElems = 32 * VEC * J;
    constexpr int kTile = WARPS * kWarpElems;
    using Acc = Access<T, VEC, true>;

    __shared__ unsigned s_tile, s_tag;
    __shared__ long long s_q0, s_r0;
    __shared__ Pair s_warp[WARPS];
    __shared__ float s_hin;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;

    // Tile ids come from a ticket so that every predecessor tile is already running
    // when its successor looks back (forward progress without relying on block order).
    if (threadIdx.x == 0) {
        const unsigned tk = atomicAdd(&ctrl->ticket, 1u);
        const long long b = static_cast<long long>(tk) * kTile;
        s_tile = tk;
        s_tag = (*reinterpret_cast<volatile unsigned*>(&ctrl->epoch) + 1u) & 0x3fffffffu;
        s_q0 = b / L;
        s_r0 = b % L;
    }
    __syncthreads();
    const unsigned tile = s_tile;
    const unsigned tag = s_tag;
    const long long base = static_cast<long long>(tile) * kTile;
    const long long q0 = s_q0, r0 = s_r0;

    TileRegs<VEC, J> r;
    // ---- A1: loads (all J vectors issued before first use)
#pragma unroll
    for (int j = 0; j < J; ++j) {
        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
        if (base + off < total) {
            Acc::load(a + base + off, r.av[j]);
            Acc::load(u + base + off, r.uv[j]);
        } else {  // identity padding (Q3)
#pragma unroll
            for (int k = 0; k < VEC; ++k) { r.av[j][k] = 1.0f; r.uv[j][k] = 0.0f; }
        }
    }
    // ---- sequence heads -> reset pairs; A4 + A5
#pragma unroll
    for (int j = 0; j < J; ++j) {
        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
        long long s, t;
        seq_pos(q0, r0, off, L, kTile, s, t);
        if (t == 0 && base + off < total) {
            const float hin = h0 ? __ldg(h0 + s) : 0.0f;
            r.uv[j][0] = fmaf(r.av[j][0], hin, r.uv[j][0]);
            r.av[j][0] = 0.0f;
        }
        row_scan(r, j, lane);
    }
    // ---- A6: cross-warp combine through shared memory
    const Pair wt = warp_total(r);
    if (lane == 0) s_warp[warp] = wt;
    __syncthreads();
    Pair X = identity_pair();  // composition of warps < warp
    for (int w = 0; w < warp; ++w) X = compose(s_warp[w], X);

    // ---- A7: decoupled look-back (warp 0)
    if (warp == 0) {
        Pair agg = s_warp[0];
#pragma unroll
        for (int w = 1; w < WARPS; ++w) agg = compose(s_warp[w], agg);
        const float h_in = lookback_carry(desc, tile, tag, agg, r0 != 0, lane);
        if (lane == 0) s_hin = h_in;
    }
    __syncthreads();

    // ---- A8: apply the prefix and rescan the thread's steps; store h, h_last
    float H = apply(X, s_hin);  // state entering this warp's slice
#pragma unroll
    for (int j = 0; j < J; ++j) {
        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
        float hs = apply(r.excl[j], H);
        float out[VEC];
#pragma unroll
        for (int k = 0; k < VEC; ++k) {
            hs = fmaf(r.av[j][k], hs, r.uv[j][k]);
            out[k] = hs;
        }
        if (base + off < total) {
            Acc::store(h + base + off, out);
            if (h_last) {
                long long s, t;
                seq_pos(q0, r0, off, L, kTile, s, t);
                if (t + VEC == L) h_last[s] = hs;
            }
        }
        H = apply(r.tot[j], H);
    }
    // The last tile to finish re-arms the control block for the next launch on this buffer.
    // Every other tile has published its INCLUSIVE descriptor before it counts itself done
    // (the barrier above orders warp 0's store before thread 0's atomic).
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned ntiles = gridDim.x;
        if (atomicAdd(&ctrl->done, 1u) == ntiles - 1) {
            ctrl->ticket = 0;
            ctrl->done = 0;
            ctrl->epoch = tag;  // = old epoch + 1 (mod 2^30)
            __threadfence();
        }
    }
}

// ====================================================================================
// Variant AFFINESCAN_AFFINE_LOOKBACK, vector path: PERSISTENT single-pass chained scan.
// Same tiles, descriptors and look-back as the kernel above, but a CTA lives for the whole
// launch: a producer warp draws tile tickets and streams the a/u tiles into a STAGES-deep
// shared-memory ring with TMA bulk copies (cp.async.bulk + mbarrier complete_tx), so the
// HBM read stream never waits for a ticket, a barrier or a look-back.  The WARPS consumer
// warps run a two-deep software pipeline over the CTA's tiles:
//     A(i+1): tile i+1 from the ring -> registers, thread/warp/CTA scan, PUBLISH its descriptor
//     B(i)  : look back for tile i (the only wait), re-read a/u of tile i from its ring slot,
//             apply the prefix, store h with 128-bit streaming stores, free the slot
// A CTA therefore never sits in a look-back wait with a tile whose aggregate its successors
// need still unpublished (a persistent CTA that waited first was measured 1.6x slower than
// the non-persistent kernel).  Between A and B a tile keeps only its 2*J prefix pairs in
// registers; its a/u stay in shared memory.
// Tickets are handed out in increasing order to running CTAs and a CTA works through its
// tiles in that order, so the smallest unfinished tile is always somebody's oldest tile with
// every predecessor finished: forward progress needs no assumption about residency.  The
// control block is re-armed by the last CTA to exit (every producer has drawn its
// terminating ticket by then).
// ====================================================================================
template <typename T, int VEC, int J, int WARPS, int STAGES>
struct ChainSmem {
    static constexpr int kTile = WARPS * 32 * VEC * J;
    static constexpr int kArrayBytes = kTile * static_cast<int>(sizeof(T));
    static constexpr int kStageBytes = 2 * kArrayBytes;  // a tile then u tile
    static constexpr int kCtrlOffset = STAGES * kStageBytes;
    // full[STAGES], empty[STAGES] mbarriers; tile id, q0, r0 per stage; s_warp[3][WARPS]; s_hin
    static constexpr int kBytes = kCtrlOffset + STAGES * 5 * 8 + 3 * WARPS * 8 + 16;
};

// First half of the look-back: publish the tile's own descriptor (no waiting).
__device__ __forceinline__ bool lookback_publish(unsigned long long* __restrict__ desc,
                                                 unsigned tile, unsigned tag, Pair agg,
                                                 bool need_carry, int lane)
{
    const bool self_contained = (agg.P == 0.0f) || !need_carry;
    if (lane == 0) {
        unsigned long long* my = desc + 2ull * tile;
        if (self_contained) desc_store(my, tag, kDescInclusive, Pair{0.0f, agg.U});
        else desc_store(my, tag, kDescAggregate, agg);
    }
    return self_contained;
}

// Second half: walk the predecessors until an INCLUSIVE one, publish INCLUSIVE, return h_in.
__device__ __forceinline__ float lookback_wait(unsigned long long* __restrict__ desc,
                                               unsigned tile, unsigned tag, Pair agg,
                                               bool self_contained, int lane)
{
    Pair acc = identity_pair();  // (+) of the tiles examined so far (later side)
    long long look = static_cast<long long>(tile) - 1;
    while (true) {
        const long long idx = look - lane;
        Pair e{0.0f, 0.0f};
        unsigned st = kDescInclusive;  // before the stream: state 0
        if (idx >= 0) {
            const unsigned long long* d = desc + 2ull * idx;
            st = desc_load(d, tag, e);
            while (st == kDescEmpty) {
                __nanosleep(32);
                st = desc_load(d, tag, e);
            }
        }
        __syncwarp();
        const unsigned incl = __ballot_sync(kFullMask, st == kDescInclusive);
        const int first = incl ? (__ffs(incl) - 1) : 32;
        if (lane > first) e = identity_pair();
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const Pair o = shfl_down_pair(e, d);
            if (lane + d < 32) e = compose(e, o);
        }
        acc = compose(acc, shfl_pair(e, 0));
        if (incl) break;
        look -= 32;
    }
    const float h_in = acc.U;  // acc.P == 0: the chain ended at an inclusive (left-zero) pair
    if (lane == 0 && !self_contained)
        desc_store(desc + 2ull * tile, tag, kDescInclusive, Pair{0.0f, apply(agg, h_in)});
    return h_in;
}

template <typename T, int VEC, int J, int WARPS, int STAGES, int CTAS_PER_SM>
__global__ void __launch_bounds__((WARPS + 1) * 32, CTAS_PER_SM)
affine_scan_chain_kernel(const T* __restrict__ a, const T* __restrict__ u,
                         const float* __restrict__ h0, T* __restrict__ h,
                         float* __restrict__ h_last, long long total, long long L,
                         long long ntiles, unsigned long long* __restrict__ desc,
                         LookbackCtrl* __restrict__ ctrl)
{
    using S = ChainSmem<T, VEC, J, WARPS, STAGES>;
    constexpr int kWarpElems = 32 * VEC * J;
    constexpr int kTile = S::kTile;
    using Acc = Access<T, VEC, true>;
    static_assert(STAGES >= 3, "a slot is held for two iterations");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + S::kCtrlOffset);
    uint64_t* empty = full + STAGES;
    long long* s_tile = reinterpret_cast<long long*>(empty + STAGES);
    long long* s_q0 = s_tile + STAGES;
    long long* s_r0 = s_q0 + STAGES;
    Pair* s_warp = reinterpret_cast<Pair*>(s_r0 + STAGES);  // [3][WARPS]
    float* s_hin = reinterpret_cast<float*>(s_warp + 3 * WARPS);

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const unsigned tag = (*reinterpret_cast<volatile unsigned*>(&ctrl->epoch) + 1u) & 0x3fffffffu;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], WARPS);
        }
        fence_mbar_init();
    }
    __syncthreads();

    if (warp == WARPS) {
        // ------------------------------------------------------------ producer warp
        if (lane == 0) {
            for (unsigned it = 0;; ++it) {
                const int st = static_cast<int>(it % STAGES);
                if (it >= STAGES) {
                    mbar_wait(&empty[st], ((it / STAGES) - 1u) & 1u);
                    // the consumers read this slot through the generic proxy; order those reads
                    // before the async-proxy overwrite below
                    fence_proxy_async_smem();
                }
                const long long tk = static_cast<long long>(atomicAdd(&ctrl->ticket, 1u));
                if (tk >= ntiles) {
                    s_tile[st] = -1;
                    mbar_arrive(&full[st]);
                    break;
                }
                const long long base = tk * kTile;
                s_tile[st] = tk;
                s_q0[st] = base / L;
                s_r0[st] = base % L;
                const long long left = total - base;
                const unsigned bytes =
                    static_cast<unsigned>(left < kTile ? left : kTile) * sizeof(T);
                unsigned char* dst = smem_raw + st * S::kStageBytes;
                mbar_arrive_expect_tx(&full[st], 2u * bytes);
                tma_bulk_g2s(dst, a + base, bytes, &full[st]);
                tma_bulk_g2s(dst + S::kArrayBytes, u + base, bytes, &full[st]);
            }
        }
    } else {
        // ------------------------------------------------------------ consumer warps
        // Short sequences that divide the tile: every tile starts at a head (no carry between
        // tiles) and a thread's vectors sit at the same place of a sequence in every tile, so the
        // head / tail flags and the sequence index inside the tile are computed once.
        const bool aligned_seq = L < kTile && (kTile % static_cast<int>(L)) == 0;
        unsigned seqmeta = 0;          // bit j: vector j starts a sequence; bit 8 + j: it ends one
        unsigned slocp[(J + 1) / 2];   // sequence index inside the tile of vector j, 16 bits each
#pragma unroll
        for (int j = 0; j < (J + 1) / 2; ++j) slocp[j] = 0;
#pragma unroll
        for (int j = 0; j < J; ++j) {
            if (aligned_seq) {
                const unsigned off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
                const unsigned Lu = static_cast<unsigned>(L);
                const unsigned sl = off / Lu;
                const unsigned t = off - sl * Lu;
                slocp[j / 2] |= sl << (16 * (j & 1));
                if (t == 0) seqmeta |= 1u << j;
                if (t + VEC == Lu) seqmeta |= 1u << (8 + j);
            }
        }
        auto sloc_of = [&](int j) { return static_cast<int>((slocp[j / 2] >> (16 * (j & 1))) & 0xffffu); };
        // state of the tile between its A and B phases
        Pair p_excl[J], p_tot[J];
        long long p_tile = -1, p_q0 = 0, p_r0 = 0;
        int p_st = 0, p_buf = 0;
        Pair p_agg = identity_pair();  // warp 0 only
        bool p_self = false;           // warp 0 only

        for (unsigned it = 0;; ++it) {
            const int st = static_cast<int>(it % STAGES);
            const int buf = static_cast<int>(it % 3);
            mbar_wait(&full[st], (it / STAGES) & 1u);
            const long long tile = s_tile[st];
            const bool cur = tile >= 0;
            const long long base = tile * kTile;
            const long long q0 = s_q0[st], r0 = s_r0[st];
            Pair c_excl[J], c_tot[J];
            if (cur) {
                // ---- A(it): ring -> registers, heads -> reset pairs, A4 + A5
                const T* sa = reinterpret_cast<const T*>(smem_raw + st * S::kStageBytes);
                const T* su = sa + kTile;
                TileRegs<VEC, J> r;
                // interior tile (the common case): whole tile inside one sequence and inside the
                // stream, so a head can only sit at offset 0 and a tail at the tile's end
                const bool fast = (r0 + kTile <= L) && (base + kTile <= total);
                if (aligned_seq && base + kTile <= total) {
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
                        unpack128<T>(*reinterpret_cast<const uint4*>(sa + off), r.av[j]);
                        unpack128<T>(*reinterpret_cast<const uint4*>(su + off), r.uv[j]);
                        if ((seqmeta >> j) & 1u) {
                            const float hin = h0 ? __ldg(h0 + q0 + sloc_of(j)) : 0.0f;
                            r.uv[j][0] = fmaf(r.av[j][0], hin, r.uv[j][0]);
                            r.av[j][0] = 0.0f;
                        }
                    }
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        row_scan(r, j, lane);
                        c_excl[j] = r.excl[j];
                        c_tot[j] = r.tot[j];
                    }
                } else if (fast) {
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
                        unpack128<T>(*reinterpret_cast<const uint4*>(sa + off), r.av[j]);
                        unpack128<T>(*reinterpret_cast<const uint4*>(su + off), r.uv[j]);
                    }
                    if (r0 == 0 && threadIdx.x == 0) {
                        const float hin = h0 ? __ldg(h0 + q0) : 0.0f;
                        r.uv[0][0] = fmaf(r.av[0][0], hin, r.uv[0][0]);
                        r.av[0][0] = 0.0f;
                    }
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        row_scan(r, j, lane);
                        c_excl[j] = r.excl[j];
                        c_tot[j] = r.tot[j];
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
                        if (base + off < total) {
                            unpack128<T>(*reinterpret_cast<const uint4*>(sa + off), r.av[j]);
                            unpack128<T>(*reinterpret_cast<const uint4*>(su + off), r.uv[j]);
                        } else {  // identity padding (Q3)
#pragma unroll
                            for (int k = 0; k < VEC; ++k) { r.av[j][k] = 1.0f; r.uv[j][k] = 0.0f; }
                        }
                    }
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
                        long long s, t;
                        seq_pos(q0, r0, off, L, kTile, s, t);
                        if (t == 0 && base + off < total) {
                            const float hin = h0 ? __ldg(h0 + s) : 0.0f;
                            r.uv[j][0] = fmaf(r.av[j][0], hin, r.uv[j][0]);
                            r.av[j][0] = 0.0f;
                        }
                        row_scan(r, j, lane);
                        c_excl[j] = r.excl[j];
                        c_tot[j] = r.tot[j];
                    }
                }
                const Pair wt = warp_total(r);
                if (lane == 0) s_warp[buf * WARPS + warp] = wt;
            }
            asm volatile("bar.sync 1, %0;" ::"n"(WARPS * 32) : "memory");
            Pair c_agg = identity_pair();
            bool c_self = false;
            if (warp == 0) {
                if (cur) {  // A6/A7: CTA aggregate, published before any waiting
                    const Pair* sw = s_warp + buf * WARPS;
                    c_agg = sw[0];
#pragma unroll
                    for (int w = 1; w < WARPS; ++w) c_agg = compose(sw[w], c_agg);
                    c_self = lookback_publish(desc, static_cast<unsigned>(tile), tag, c_agg,
                                              r0 != 0, lane);
                }
                if (p_tile >= 0) {  // the only wait: carry into the previous tile
                    float h_in = 0.0f;
                    if (p_r0 != 0)
                        h_in = lookback_wait(desc, static_cast<unsigned>(p_tile), tag, p_agg,
                                             p_self, lane);
                    if (lane == 0) *s_hin = h_in;
                }
            }
            asm volatile("bar.sync 1, %0;" ::"n"(WARPS * 32) : "memory");
            if (p_tile >= 0) {
                // ---- B(it-1): apply the prefix, rescan from the ring slot, store h, h_last
                const Pair* sw = s_warp + p_buf * WARPS;
                Pair X = identity_pair();
                for (int w = 0; w < warp; ++w) X = compose(sw[w], X);
                float H = apply(X, *s_hin);
                const long long pbase = p_tile * kTile;
                const T* sa = reinterpret_cast<const T*>(smem_raw + p_st * S::kStageBytes);
                const T* su = sa + kTile;
                const bool fast = (p_r0 + kTile <= L) && (pbase + kTile <= total);
                if (aligned_seq && pbase + kTile <= total) {
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
                        float av[VEC], uv[VEC];
                        unpack128<T>(*reinterpret_cast<const uint4*>(sa + off), av);
                        unpack128<T>(*reinterpret_cast<const uint4*>(su + off), uv);
                        float hs = apply(p_excl[j], H);
                        if ((seqmeta >> j) & 1u) hs = h0 ? __ldg(h0 + p_q0 + sloc_of(j)) : 0.0f;
                        float out[VEC];
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            hs = fmaf(av[k], hs, uv[k]);
                            out[k] = hs;
                        }
                        Acc::store(h + pbase + off, out);
                        if (((seqmeta >> (8 + j)) & 1u) && h_last) h_last[p_q0 + sloc_of(j)] = hs;
                        H = apply(p_tot[j], H);
                    }
                } else if (fast) {
                    const bool tail = (p_r0 + kTile == L);
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
                        float av[VEC], uv[VEC];
                        unpack128<T>(*reinterpret_cast<const uint4*>(sa + off), av);
                        unpack128<T>(*reinterpret_cast<const uint4*>(su + off), uv);
                        float hs = apply(p_excl[j], H);
                        if (j == 0 && p_r0 == 0 && threadIdx.x == 0) hs = h0 ? __ldg(h0 + p_q0) : 0.0f;
                        float out[VEC];
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            hs = fmaf(av[k], hs, uv[k]);
                            out[k] = hs;
                        }
                        Acc::store(h + pbase + off, out);
                        if (j == J - 1 && tail && h_last && threadIdx.x == WARPS * 32 - 1)
                            h_last[p_q0] = hs;
                        H = apply(p_tot[j], H);
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        const int off = warp * kWarpElems + j * 32 * VEC + lane * VEC;
                        if (pbase + off < total) {
                            float av[VEC], uv[VEC];
                            unpack128<T>(*reinterpret_cast<const uint4*>(sa + off), av);
                            unpack128<T>(*reinterpret_cast<const uint4*>(su + off), uv);
                            long long s, t;
                            seq_pos(p_q0, p_r0, off, L, kTile, s, t);
                            float hs = apply(p_excl[j], H);
                            if (t == 0) hs = h0 ? __ldg(h0 + s) : 0.0f;  // head: the reset pair
                            float out[VEC];
#pragma unroll
                            for (int k = 0; k < VEC; ++k) {
                                hs = fmaf(av[k], hs, uv[k]);
                                out[k] = hs;
                            }
                            Acc::store(h + pbase + off, out);
                            if (h_last && t + VEC == L) h_last[s] = hs;
                        }
                        H = apply(p_tot[j], H);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[p_st]);  // the slot may be refilled
            }
            if (!cur) break;
#pragma unroll
            for (int j = 0; j < J; ++j) { p_excl[j] = c_excl[j]; p_tot[j] = c_tot[j]; }
            p_tile = tile; p_q0 = q0; p_r0 = r0; p_st = st; p_buf = buf;
            p_agg = c_agg; p_self = c_self;
        }
    }
    // The last CTA to exit re-arms the control block for the next launch on this buffer.
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&ctrl->done, 1u) == gridDim.x - 1) {
            ctrl->ticket = 0;
            ctrl->done = 0;
            ctrl->epoch = tag;  // = old epoch + 1 (mod 2^30)
            __threadfence();
        }
    }
}

// ====================================================================================
// Variant AFFINESCAN_AFFINE_CTA_LOOP: one CTA per sequence, carry in a register (A7-i)
// ====================================================================================
template <typename T, int VEC, int J, int WARPS>
__global__ void __launch_bounds__(WARPS * 32)
affine_scan_cta_loop_kernel(const T* __restrict__ a, const T* __restrict__ u,
                            const float* __restrict__ h0, T* __restrict__ h,
                            float* __restrict__ h_last, long long num_seq, long long L)
{
    constexpr int kWarpElems = 32 * VEC * J;
    constexpr int kTile = WARPS * kWarpElems;
    using Acc = Access<T, VEC, true>;
    __shared__ Pair s_warp[2][WARPS];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;

    for (long long s = blockIdx.x; s < num_seq; s += gridDim.x) {
        const T* as = a + s * L;
        const T* us = u + s * L;
        T* hs_out = h + s * L;
        float carry = h0 ? __ldg(h0 + s) : 0.0f;
        int buf = 0;
        for (long long t0 = 0; t0 < L; t0 += kTile, buf ^= 1) {
            TileRegs<VEC, J> r;
#pragma unroll
            for (int j = 0; j < J; ++j) {
                const long long t = t0 + warp * kWarpElems + j * 32 * VEC + lane * VEC;
                if (t < L) {
                    Acc::load(as + t, r.av[j]);
                    Acc::load(us + t, r.uv[j]);
                } else {
#pragma unroll
                    for (int k = 0; k < VEC; ++k) { r.av[j][k] = 1.0f; r.uv[j][k] = 0.0f; }
                }
            }
#pragma unroll
            for (int j = 0; j < J; ++j) row_scan(r, j, lane);
            Pair X = identity_pair();
            Pair agg = warp_total(r);
            if (WARPS > 1) {
                if (lane == 0) s_warp[buf][warp] = agg;
                __syncthreads();  // one barrier per tile: s_warp is double-buffered
                agg = s_warp[buf][0];
#pragma unroll
                for (int w = 1; w < WARPS; ++w) {
                    if (w == warp) X = agg;
                    agg = compose(s_warp[buf][w], agg);
                }
            }
            float H = apply(X, carry);
#pragma unroll
            for (int j = 0; j < J; ++j) {
                const long long t = t0 + warp * kWarpElems + j * 32 * VEC + lane * VEC;
                float hv = apply(r.excl[j], H);
                float out[VEC];
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    hv = fmaf(r.av[j][k], hv, r.uv[j][k]);
                    out[k] = hv;
                }
                if (t < L) {
                    Acc::store(hs_out + t, out);
                    // h_last is the very value stored at t = L-1 (bitwise)
                    if (h_last && t + VEC >= L) h_last[s] = hv;
                }
                H = apply(r.tot[j], H);
            }
            carry = apply(agg, carry);
        }
    }
}

// ====================================================================================
// Variant AFFINESCAN_AFFINE_WARP_SEQ: one WARP per sequence (many short sequences), carry in a
// register (A7-i), no shared memory and no barrier: warps of a CTA are independent.
// ====================================================================================
template <typename T, int VEC, int J, int WARPS>
__global__ void __launch_bounds__(WARPS * 32)
affine_scan_warp_seq_kernel(const T* __restrict__ a, const T* __restrict__ u,
                            const float* __restrict__ h0, T* __restrict__ h,
                            float* __restrict__ h_last, long long num_seq, long long L)
{
    constexpr int kWarpElems = 32 * VEC * J;
    using Acc = Access<T, VEC, true>;
    const int lane = threadIdx.x & 31;
    const long long gwarp = static_cast<long long>(blockIdx.x) * WARPS + (threadIdx.x >> 5);
    const long long nwarps = static_cast<long long>(gridDim.x) * WARPS;

    for (long long s = gwarp; s < num_seq; s += nwarps) {
        const T* as = a + s * L;
        const T* us = u + s * L;
        T* hs_out = h + s * L;
        float carry = h0 ? __ldg(h0 + s) : 0.0f;
        for (long long t0 = 0; t0 < L; t0 += kWarpElems) {
            TileRegs<VEC, J> r;
#pragma unroll
            for (int j = 0; j < J; ++j) {
                const long long t = t0 + j * 32 * VEC + lane * VEC;
                if (t < L) {
                    Acc::load(as + t, r.av[j]);
                    Acc::load(us + t, r.uv[j]);
                } else {
#pragma unroll
                    for (int k = 0; k < VEC; ++k) { r.av[j][k] = 1.0f; r.uv[j][k] = 0.0f; }
                }
            }
#pragma unroll
            for (int j = 0; j < J; ++j) row_scan(r, j, lane);
            float H = carry;
#pragma unroll
            for (int j = 0; j < J; ++j) {
                const long long t = t0 + j * 32 * VEC + lane * VEC;
                float hv = apply(r.excl[j], H);
                float out[VEC];
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    hv = fmaf(r.av[j][k], hv, r.uv[j][k]);
                    out[k] = hv;
                }
                if (t < L) {
                    Acc::store(hs_out + t, out);
                    if (h_last && t + VEC >= L) h_last[s] = hv;  // the value stored at t = L-1
                }
                H = apply(r.tot[j], H);
            }
            carry = H;
        }
    }
}

// ====================================================================================
// Variant AFFINESCAN_AFFINE_BLELLOCH (ABLATION): the paper's schedule (P:103-107,
// P:163-167; Q3/Q4/Q16) on a shared-memory tile of 2*THREADS pairs:
// upsweep (tree reduction), root <- (1,0), downsweep (prefix propagation), affine-prefix
// reconstruction incl_t = e_t (+) excl_t, h_t = A_incl*carry + U_incl; CTA-loop carry.
// Deliberately textbook: 2*log2(tile) barriers per tile and strided (bank-conflicting)
// tree accesses are exactly the overheads the paper names.
// ====================================================================================
template <typename T, int THREADS>
__global__ void __launch_bounds__(THREADS)
affine_scan_blelloch_kernel(const T* __restrict__ a, const T* __restrict__ u,
                            const float* __restrict__ h0, T* __restrict__ h,
                            float* __restrict__ h_last, long long num_seq, long long L)
{
    constexpr int kTile = 2 * THREADS;
    using Acc = Access<T, 1, false>;
    __shared__ float sP[kTile];
    __shared__ float sU[kTile];
    __shared__ Pair s_total;
    const int tid = threadIdx.x;

    for (long long s = blockIdx.x; s < num_seq; s += gridDim.x) {
        const T* as = a + s * L;
        const T* us = u + s * L;
        T* ho = h + s * L;
        float carry = h0 ? __ldg(h0 + s) : 0.0f;
        for (long long t0 = 0; t0 < L; t0 += kTile) {
            float ea[2], eu[2];
#pragma unroll
            for (int i = 0; i < 2; ++i) {  // shared-memory staging of the pairs
                const long long t = t0 + tid + i * THREADS;
                float va[1] = {1.0f}, vu[1] = {0.0f};  // identity padding (Q3)
                if (t < L) { Acc::load(as + t, va); Acc::load(us + t, vu); }
                ea[i] = va[0]; eu[i] = vu[0];
                sP[tid + i * THREADS] = ea[i];
                sU[tid + i * THREADS] = eu[i];
            }
            // upsweep: x[r] <- x[r] (+) x[l], r later
            for (int stride = 1; stride < kTile; stride <<= 1) {
                __syncthreads();
                const int rr = (tid + 1) * 2 * stride - 1;
                if (rr < kTile) {
                    const int ll = rr - stride;
                    const Pair v = compose(Pair{sP[rr], sU[rr]}, Pair{sP[ll], sU[ll]});
                    sP[rr] = v.P; sU[rr] = v.U;
                }
            }
            __syncthreads();
            if (tid == 0) {  // root initialisation: keep the total, root <- identity
                s_total = Pair{sP[kTile - 1], sU[kTile - 1]};
                sP[kTile - 1] = 1.0f; sU[kTile - 1] = 0.0f;
            }
            // downsweep: t <- x[l]; x[l] <- x[r]; x[r] <- t (+) x[r]_old
            for (int stride = kTile >> 1; stride >= 1; stride >>= 1) {
                __syncthreads();
                const int rr = (tid + 1) * 2 * stride - 1;
                if (rr < kTile) {
                    const int ll = rr - stride;
                    const Pair left{sP[ll], sU[ll]};
                    const Pair inh{sP[rr], sU[rr]};
                    sP[ll] = inh.P; sU[ll] = inh.U;
                    const Pair v = compose(left, inh);
                    sP[rr] = v.P; sU[rr] = v.U;
                }
            }
            __syncthreads();
            // affine-prefix reconstruction
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int idx = tid + i * THREADS;
                const long long t = t0 + idx;
                const Pair incl = compose(Pair{ea[i], eu[i]}, Pair{sP[idx], sU[idx]});
                float out[1] = {apply(incl, carry)};
                if (t < L) Acc::store(ho + t, out);
            }
            carry = apply(s_total, carry);
            __syncthreads();  // smem tile and s_total are reused by the next tile
        }
        if (h_last && tid == 0) h_last[s] = carry;
    }
}

}  // namespace affinescan
