// selective_scan_warp_row_tma.cuh — variant AFFINESCAN_SELECTIVE_WARP_ROW_TMA of
// selective_scan_fwd (include/affinescan.h; BJ north_star).
//
// The few-rows schedule (cfg2, cfg4: 1536 rows): the scan over L is parallelised inside the
// warp.  One warp owns one (b,d) row; a warp tile is 32*K consecutive timesteps, lane l owning
// the K consecutive steps [l*K, l*K+K).  A CTA is R warps = R rows of ONE batch, so B_t/C_t
// are shared by the whole CTA: an elected thread stages the [N][32*K] tiles of B and of C with
// TMA tensor copies (cp.async.bulk.tensor.2d, boxes of 128/256 timesteps x N rows, mbarrier
// complete_tx) into a 2-stage shared-memory ring; the elected thread lives in a dedicated
// producer warp; consumers release a stage through an "empty" mbarrier (one arrival per warp).
// For each state n (outer loop, NU states per iteration for ILP) a lane
//   A3  discretises      a_k = ex2(delta_k * A2[n]),  u_k = (delta_k x_k) * B_k[n]   (smem)
//   A4  composes its K pairs in registers (P via one ex2 of A2[n]*sum(delta))
//   A5  combines across the warp with a Kogge–Stone __shfl_up_sync pair scan
//   A7  takes the carry h_in[n] of the previous tile (register, CTA-loop style)
//   A8  rescans its K steps from the exclusive prefix (a_k, u_k still in registers)
//   A9  accumulates y_k += C_k[n] * h_k (smem) ; h itself is never stored.
// x/delta/y move with coalesced 128-bit global accesses (lane owns K contiguous elements).
//
// Template mode LB = variant AFFINESCAN_SELECTIVE_CHUNKED (BJ "decoupled
// look-back for very long sequences"): the same tile body, but the (tile, row-block) work items
// are handed out tile-major by an atomic ticket to persistent CTAs, so L is parallelised across
// CTAs and occupancy no longer depends on the row count.  The carry h_in[n] of a tile is no
// longer a register of the warp that ran the previous tile.  Per (row, tile):
//   phase A   the tile's aggregate pair (P, U) of every state (discretise, local compose, ordered
//             warp reduction; the a_k, u_k are NOT kept) is published as one descriptor per state;
//   look-back ONE decoupled look-back for all N states: lane = predecessor tile (32 at a time),
//             the descriptors of every state are requested before any is consumed (one L2 round
//             trip per window), each state's window is folded with an ordered shuffle tree and
//             stops at its first INCLUSIVE descriptor; then INCLUSIVE (0, h_out) is published;
//   phase B   the plain tile body with h_in as the carry (the 2^x are recomputed: the schedule
//             pays a second exp per state-step to break the serial chain over tiles, and is
//             chosen only when rows are too few to fill the machine otherwise).
// Descriptors are epoch-tagged: nothing is cleared per call.
#pragma once

#include <type_traits>

#include "affine_scan.cuh"  // tile descriptors of the decoupled look-back
#include "selective_common.cuh"
#include "tma.cuh"

namespace affinescan {

// Decoupled look-back for ALL N states of (row, tile) at once (LB mode).  `drow` = descriptors of
// this row, [ntiles][N][2] 64-bit words; lane n < N holds the tile's aggregate (totP, totU) of
// state n and h0n = h0[n].  Returns on lane n the carry-in h_in[n]; publishes AGGREGATE then
// INCLUSIVE (0, h_out) per state.  Lanes are predecessor tiles while looking back.
template <int N>
__device__ __forceinline__ float selective_lookback_all(unsigned long long* drow, long long tile,
                                                        unsigned tag, float totP, float totU,
                                                        float h0n, int lane)
{
    unsigned long long* my = drow + (tile * N + lane) * 2;
    if (tile == 0) {
        if (lane < N) desc_store(my, tag, kDescInclusive, Pair{0.0f, fmaf(totP, h0n, totU)});
        return h0n;
    }
    // P == 0 (underflow, or a reset inside the tile): the state after the tile does not depend
    // on the carry, so successors need not wait for ours — but this tile's own early steps do
    const bool self_contained = totP == 0.0f;
    if (lane < N) {
        if (self_contained) desc_store(my, tag, kDescInclusive, Pair{0.0f, totU});
        else desc_store(my, tag, kDescAggregate, Pair{totP, totU});
    }
    Pair acc = identity_pair();        // lane n: (+) of the tiles examined so far for state n
    unsigned pending = (1u << N) - 1;  // states whose chain has not reached an INCLUSIVE yet
    long long look = tile - 1;
    while (pending) {
        const long long idx = look - lane;
        Pair e[N];
        unsigned st[N];
        // request every pending state's descriptor of this lane's tile before consuming any
#pragma unroll
        for (int n = 0; n < N; ++n) {
            e[n] = Pair{0.0f, 0.0f};
            st[n] = kDescInclusive;  // before tile 0: never selected (tile 0 is INCLUSIVE)
            if (((pending >> n) & 1u) && idx >= 0) st[n] = desc_load(drow + (idx * N + n) * 2, tag, e[n]);
        }
#pragma unroll
        for (int n = 0; n < N; ++n) {
            if (!((pending >> n) & 1u)) continue;  // warp-uniform
            if (idx >= 0) {
                while (st[n] == kDescEmpty) {
                    __nanosleep(20);
                    st[n] = desc_load(drow + (idx * N + n) * 2, tag, e[n]);
                }
            }
            __syncwarp();
            const unsigned incl = __ballot_sync(kFullMask, st[n] == kDescInclusive);
            const int first = incl ? (__ffs(incl) - 1) : 32;
            Pair w = lane > first ? identity_pair() : e[n];
            // ordered tree reduction: lane 0 holds the LATEST tile (left operand of (+))
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const Pair o = shfl_down_pair(w, d);
                if (lane + d < 32) w = compose(w, o);
            }
            const Pair win = shfl_pair(w, 0);
            if (lane == n) acc = compose(acc, win);
            if (incl) pending &= ~(1u << n);
        }
        // a chain whose accumulated product has underflowed to exactly 0 is finished too: every
        // earlier tile would be multiplied by that 0 (Q18), so nothing is approximated
        pending &= ~__ballot_sync(kFullMask, lane < N && acc.P == 0.0f);
        look -= 32;
    }
    const float h_in = acc.U;  // acc.P == 0: an inclusive (left-zero) pair, or underflow
    if (lane < N && !self_contained)
        desc_store(my, tag, kDescInclusive, Pair{0.0f, fmaf(totP, h_in, totU)});
    return h_in;
}

template <typename T, int K>
struct WarpRowTmaSmem {
    static constexpr int N = 16;
    static constexpr int kTileT = 32 * K;                    // timesteps per warp tile
    static constexpr int kNv = K * static_cast<int>(sizeof(T)) / 16;  // 128-bit vectors per lane
    static constexpr int kBoxT = kTileT / kNv;               // TMA box: <= 256 elements per dim
    static constexpr int kBoxes = kTileT / kBoxT;            // boxes per tensor per tile
    static constexpr int kBoxBytes = N * kBoxT * static_cast<int>(sizeof(T));
    static constexpr int kStageBytes = 2 * kBoxes * kBoxBytes;  // B boxes then C boxes
    static constexpr int kStages = 2;
    static constexpr int kBytes = kStages * kStageBytes + 64;   // + full[2], empty[2], item[2]
    static_assert(kTileT % kBoxT == 0 && kBoxT <= 256, "tile is a whole number of boxes");
    // Bank conflicts: lane l reads the 16-byte chunks l*NV + v (v < NV) of a row.  Box and row
    // strides are multiples of 128 B, so the 8 lanes of an LDS.128 phase hit distinct 16-byte
    // slots iff NV is odd (K = 12 for fp32 io, 24 for bf16 io).
    static_assert((K * sizeof(T) / 16) % 2 == 1, "odd number of 128-bit vectors per lane");
    static_assert((kBoxT * sizeof(T)) % 128 == 0, "row stride multiple of 128 B");
};

// NU = states processed together per n-iteration (independent chains per warp).
// EXT = the fused steps either side of the scan (softplus/bias, silu(z) gate, resets).
// LB  = ticketed (tile, row-block) work items with the decoupled look-back carry (CHUNKED).
template <typename T, int VEC, int NV, int NU, bool EXT, bool LB>
__global__ void __launch_bounds__(384, 1)
selective_scan_warp_row_tma_kernel(const T* __restrict__ x, const T* __restrict__ delta,
                                   const float* __restrict__ A,
                                   const __grid_constant__ CUtensorMap mapB,
                                   const __grid_constant__ CUtensorMap mapC,
                                   const float* __restrict__ D, const float* __restrict__ h0,
                                   T* __restrict__ y, float* __restrict__ h_last,
                                   const SelectiveExt ext, int batch, int d_inner,
                                   int ctas_per_batch, long long L,
                                   unsigned long long* __restrict__ desc,
                                   LookbackCtrl* __restrict__ ctrl)
{
    constexpr int K = NV * VEC;
    using S = WarpRowTmaSmem<T, K>;
    constexpr int N = S::N;
    using AccS = Access<T, VEC, true>;  // streamed once: x, delta, y, z

    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + S::kStages * S::kStageBytes);
    uint64_t* empty = full + S::kStages;
    long long* item_of_stage = reinterpret_cast<long long*>(empty + S::kStages);  // LB only

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int R = (blockDim.x >> 5) - 1;  // consumer warps per CTA; warp R is the producer

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < S::kStages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], static_cast<unsigned>(R));
        }
        fence_mbar_init();
    }
    fence_proxy_async_smem();
    __syncthreads();

    const long long ntiles = (L + S::kTileT - 1) / S::kTileT;
    const long long slots = static_cast<long long>(batch) * ctas_per_batch;  // row-blocks
    // steps = stage uses of this CTA: its own tiles 0..ntiles-1 (plain), or ticketed work
    // items until the producer draws a ticket past the end (LB)
    const long long nitems = LB ? ntiles * slots : ntiles;
    const unsigned tag = LB ? ((*reinterpret_cast<volatile unsigned*>(&ctrl->epoch) + 1u) & 0x3fffffffu) : 0u;

    auto issue_tile = [&](int st, long long tile, int b) {  // one thread
        unsigned char* dst = smem_raw + st * S::kStageBytes;
        mbar_arrive_expect_tx(&full[st], static_cast<unsigned>(S::kStageBytes));
#pragma unroll
        for (int i = 0; i < S::kBoxes; ++i) {
            const int t0 = static_cast<int>(tile * S::kTileT) + i * S::kBoxT;
            tma_tile_2d_g2s(dst + i * S::kBoxBytes, &mapB, t0, b * N, &full[st]);
            tma_tile_2d_g2s(dst + (S::kBoxes + i) * S::kBoxBytes, &mapC, t0, b * N, &full[st]);
        }
    };
    // Producer warp: one elected lane keeps the 2-stage ring full; it refills a stage as soon
    // as every consumer warp has released it, and never touches the data itself.  In LB mode
    // it also draws the work items: tile-major tickets, so that every predecessor tile of an
    // item is already running (or done) when its consumers look back.
    if (warp == R) {
        if (lane == 0) {
            for (long long step = 0;; ++step) {
                const int st = static_cast<int>(step % S::kStages);
                if (step >= S::kStages) {
                    const long long prev = step - S::kStages;  // the step that used this stage
                    mbar_poll(&empty[st], static_cast<unsigned>((prev / S::kStages) & 1));
                    fence_proxy_async_smem();
                }
                if (LB && step >= 1) {
                    // A drawn ticket must be worked on at once: successors of a tile that sits
                    // prefetched behind this CTA's current item would all wait for it (every
                    // look-back polls its predecessors' aggregates).  So the next ticket is drawn
                    // only when the consumers have released the PREVIOUS item; the staging
                    // latency this exposes is covered by the second CTA on the SM.
                    const long long prev = step - 1;
                    mbar_poll(&empty[prev % S::kStages], static_cast<unsigned>((prev / S::kStages) & 1));
                }
                if (LB) {
                    const long long item = atomicAdd(&ctrl->ticket, 1u);
                    if (item >= nitems) {  // no more work: wake the consumers with a stop item
                        item_of_stage[st] = -1;
                        mbar_arrive(&full[st]);
                        break;
                    }
                    item_of_stage[st] = item;
                    const long long tile = item / slots;
                    const int b = static_cast<int>((item - tile * slots) / ctas_per_batch);
                    issue_tile(st, tile, b);
                } else {
                    if (step >= ntiles) break;
                    issue_tile(st, step, blockIdx.x / ctas_per_batch);
                }
            }
        }
    } else {
        // ---------------------------------------------------------------- consumer warps
        // per-row values: reloaded per work item in LB mode, once otherwise
        int b = 0, dd = 0;
        bool active = false;
        long long row = 0;
        float A2r = 0.0f, hcr = 0.0f, Dd = 0.0f, bias = 0.0f;
        const T* zr = nullptr;
        const unsigned char* rst = nullptr;
        unsigned long long* drow = nullptr;
        auto bind_row = [&](int bb, int d0) {
            b = bb;
            // an inactive row is computed (on a valid row) but never stored or published: its
            // warp still takes part in the stage ring
            active = d0 + warp < d_inner;
            dd = active ? d0 + warp : d_inner - 1;
            row = static_cast<long long>(b) * d_inner + dd;
            // lane n keeps A2[n] = A[d,n]*log2(e) and (plain mode) the carry h_in[n] of the row
            A2r = lane < N ? __ldg(A + static_cast<long long>(dd) * N + lane) * kLog2e : 0.0f;
            hcr = (lane < N && h0) ? __ldg(h0 + row * N + lane) : 0.0f;  // LB: h0, used by tile 0
            Dd = D ? __ldg(D + dd) : 0.0f;
            bias = (EXT && ext.delta_bias) ? __ldg(ext.delta_bias + dd) : 0.0f;
            zr = (EXT && ext.z) ? static_cast<const T*>(ext.z) + row * L : nullptr;
            rst = (EXT && ext.reset) ? ext.reset + static_cast<long long>(b) * L : nullptr;
            if (LB) drow = desc + row * ntiles * N * 2;
        };
        if (!LB) {
            const int bb = blockIdx.x / ctas_per_batch;
            bind_row(bb, (blockIdx.x - bb * ctas_per_batch) * R);
        }

        // byte offset (inside a tensor's stage, state n = 0) of this lane's v-th 128-bit vector
        int voff[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const int t = lane * K + v * VEC;  // timestep inside the tile
            voff[v] = (t / S::kBoxT) * S::kBoxBytes + (t % S::kBoxT) * static_cast<int>(sizeof(T));
        }

        // A1: raw 128-bit loads of the lane's K timesteps of x and delta (plain mode: one tile ahead)
        uint4 xq[NV], dq[NV];
        auto prefetch = [&](long long tile) {
            const long long tl = tile * S::kTileT + lane * K;
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                xq[v] = make_uint4(0, 0, 0, 0);  // identity padding: delta = 0 => a = 1, u = 0 (Q12)
                dq[v] = make_uint4(0, 0, 0, 0);
                if (tl + v * VEC < L) {
                    xq[v] = __ldcs(reinterpret_cast<const uint4*>(x + row * L + tl + v * VEC));
                    dq[v] = __ldcs(reinterpret_cast<const uint4*>(delta + row * L + tl + v * VEC));
                }
            }
        };
        if (!LB) prefetch(0);

        for (long long step = 0;; ++step) {
            const int st = static_cast<int>(step % S::kStages);
            const unsigned parity = static_cast<unsigned>((step / S::kStages) & 1);
            long long tile = step;
            if (LB) {
                mbar_wait(&full[st], parity);
                const long long item = item_of_stage[st];
                if (item < 0) break;
                tile = item / slots;
                const long long rem = item - tile * slots;
                const int bb = static_cast<int>(rem / ctas_per_batch);
                bind_row(bb, static_cast<int>(rem - static_cast<long long>(bb) * ctas_per_batch) * R);
                prefetch(tile);
            } else if (step >= ntiles) {
                break;
            }
            const long long tl = tile * S::kTileT + lane * K;  // first timestep of this lane
            float dl[K], dx[K], yv[K], dsum = 0.0f;
            unsigned rmask = 0;  // bit k: timestep tl + k starts a new sequence (f2)
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                float xv[VEC], dv[VEC];
                unpack128<T>(xq[v], xv);
                unpack128<T>(dq[v], dv);
                const bool in = tl + v * VEC < L;
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    if (EXT) {  // f1 prologue; padding keeps delta = 0
                        const float t = dv[k] + bias;
                        dv[k] = in ? (ext.delta_softplus ? softplus_f(t) : t) : 0.0f;
                        if (rst && in)
                            rmask |= (__ldg(rst + tl + v * VEC + k) != 0 ? 1u : 0u) << (v * VEC + k);
                    }
                    dl[v * VEC + k] = dv[k];
                    dx[v * VEC + k] = dv[k] * xv[k];
                    yv[v * VEC + k] = Dd * xv[k];
                }
            }
#pragma unroll
            for (int k = 0; k < K; ++k) dsum += dl[k];
            if (!LB) {
                if (tile + 1 < ntiles) prefetch(tile + 1);
                mbar_wait(&full[st], parity);
            }
            const unsigned char* sB = smem_raw + st * S::kStageBytes;
            const unsigned char* sC = sB + S::kBoxes * S::kBoxBytes;

            // RST: some lane of the warp holds a reset in this tile (a_k := 0 there, and the
            // lane's chunk product P := 0: the pair of a reset step is the left zero (0, u_t) of
            // (+))
            auto states = [&](auto rtag) {
                constexpr bool RST = decltype(rtag)::value;
#pragma unroll 1
                for (int n0 = 0; n0 < N; n0 += NU) {
                    float a[NU][K], u[NU][K];
                    Pair inc[NU];
                    float hin[NU];
                    // ---- A3 + A4 for NU states: independent work, issued back to back
#pragma unroll
                    for (int j = 0; j < NU; ++j) {
                        const int n = n0 + j;
                        const float A2n = __shfl_sync(kFullMask, A2r, n);
                        hin[j] = __shfl_sync(kFullMask, hcr, n);
                        const unsigned char* bn = sB + n * S::kBoxT * static_cast<int>(sizeof(T));
#pragma unroll
                        for (int v = 0; v < NV; ++v) {
                            float bv[VEC];
                            unpack128<T>(*reinterpret_cast<const uint4*>(bn + voff[v]), bv);
#pragma unroll
                            for (int k = 0; k < VEC; ++k) {
                                float ak = ex2_approx(dl[v * VEC + k] * A2n);
                                if (RST && ((rmask >> (v * VEC + k)) & 1u)) ak = 0.0f;
                                a[j][v * VEC + k] = ak;
                                u[j][v * VEC + k] = dx[v * VEC + k] * bv[k];
                            }
                        }
                        float Pl = ex2_approx(dsum * A2n);
                        if (RST && rmask != 0) Pl = 0.0f;
                        inc[j] = Pair{Pl, u[j][0]};
                    }
#pragma unroll
                    for (int k = 1; k < K; ++k) {
#pragma unroll
                        for (int j = 0; j < NU; ++j) inc[j].U = fmaf(a[j][k], inc[j].U, u[j][k]);
                    }
                    // ---- A5: warp combine (NU interleaved Kogge–Stone scans)
#pragma unroll
                    for (int dlt = 1; dlt < 32; dlt <<= 1) {
                        Pair pv[NU];
#pragma unroll
                        for (int j = 0; j < NU; ++j) pv[j] = shfl_up_pair(inc[j], dlt);
                        if (lane >= dlt) {
#pragma unroll
                            for (int j = 0; j < NU; ++j) inc[j] = compose(inc[j], pv[j]);
                        }
                    }
                    // ---- A7/A8: carry-in, rescan; A9: y accumulation
#pragma unroll
                    for (int j = 0; j < NU; ++j) {
                        const int n = n0 + j;
                        Pair ex = shfl_up_pair(inc[j], 1);
                        if (lane == 0) ex = identity_pair();
                        const Pair tot = shfl_pair(inc[j], 31);
                        const float hout = apply(tot, hin[j]);  // state after the tile (uniform)
                        if (lane == n) hcr = hout;
                        float hv = apply(ex, hin[j]);
                        const unsigned char* cn = sC + n * S::kBoxT * static_cast<int>(sizeof(T));
#pragma unroll
                        for (int v = 0; v < NV; ++v) {
                            float cc[VEC];
                            unpack128<T>(*reinterpret_cast<const uint4*>(cn + voff[v]), cc);
#pragma unroll
                            for (int k = 0; k < VEC; ++k) {
                                hv = fmaf(a[j][v * VEC + k], hv, u[j][v * VEC + k]);
                                yv[v * VEC + k] = fmaf(cc[k], hv, yv[v * VEC + k]);
                            }
                        }
                    }
                }
            };
            const bool tile_has_reset = EXT && __any_sync(kFullMask, rmask != 0);
            if (LB) {
                // ---- phase A: the tile's aggregate pair of every state; lane n keeps state n's
                float totP = 1.0f, totU = 0.0f;
#pragma unroll 1
                for (int n = 0; n < N; ++n) {
                    const float A2n = __shfl_sync(kFullMask, A2r, n);
                    const unsigned char* bn = sB + n * S::kBoxT * static_cast<int>(sizeof(T));
                    Pair loc{ex2_approx(dsum * A2n), 0.0f};
                    if (tile_has_reset && rmask != 0) loc.P = 0.0f;
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        float bv[VEC];
                        unpack128<T>(*reinterpret_cast<const uint4*>(bn + voff[v]), bv);
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            float ak = ex2_approx(dl[v * VEC + k] * A2n);
                            if (tile_has_reset && ((rmask >> (v * VEC + k)) & 1u)) ak = 0.0f;
                            loc.U = fmaf(ak, loc.U, dx[v * VEC + k] * bv[k]);
                        }
                    }
                    const Pair inc = warp_inclusive_scan(loc, lane);
                    const Pair tot = shfl_pair(inc, 31);
                    if (lane == n) { totP = tot.P; totU = tot.U; }
                }
                // ---- A7-ii: one decoupled look-back for all states; lane n gets h_in[n].
                // Inactive rows neither publish nor look back (their row duplicates a real one).
                if (active) hcr = selective_lookback_all<N>(drow, tile, tag, totP, totU, hcr, lane);
            }
            // ---- phase B (LB) / the tile body (plain): carry in hcr, lane n holds state n's
            if (tile_has_reset) states(std::true_type{});
            else states(std::false_type{});
            if (LB && h_last && active && tile == ntiles - 1 && lane < N) h_last[row * N + lane] = hcr;
            // release the stage; the producer warp refills it once every warp has
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
            // ---- A9: store y (f1 epilogue: y <- y * silu(z))
            if (active) {
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    if (tl + v * VEC < L) {
                        float out[VEC];
#pragma unroll
                        for (int k = 0; k < VEC; ++k) out[k] = yv[v * VEC + k];
                        if (EXT && zr) {
                            float zv[VEC];
                            AccS::load(zr + tl + v * VEC, zv);
#pragma unroll
                            for (int k = 0; k < VEC; ++k) out[k] *= silu_io<T>(zv[k]);
                        }
                        if (y) AccS::store(y + row * L + tl + v * VEC, out);  // NULL: aggregate-only
                    }
                }
            }
        }
        // ---- A10: final state (plain mode: the carry register after the last tile)
        if (!LB && h_last && active && lane < N) h_last[row * N + lane] = hcr;
    }

    if (LB) {
        // The last CTA to finish re-arms the control block for the next launch on this buffer
        // (every INCLUSIVE descriptor of this launch has been published by then).
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            if (atomicAdd(&ctrl->done, 1u) == gridDim.x - 1) {
                ctrl->ticket = 0;
                ctrl->done = 0;
                ctrl->epoch = tag;
                __threadfence();
            }
        }
    }
}

}  // namespace affinescan
