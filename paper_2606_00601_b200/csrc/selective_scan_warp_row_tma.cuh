// selective_scan_warp_row_tma.cuh — variant AFFINESCAN_SELECTIVE_WARP_ROW_TMA of
// selective_scan_fwd (include/affinescan.h; BJ north_star).
//
// The few-rows schedule (cfg2, cfg4: 1536 rows): the scan over L is parallelised inside the
// warp.  One warp owns one (b,d) row; a warp tile is 32*K consecutive timesteps, lane l owning
// the K consecutive steps [l*K, l*K+K).  A CTA is R warps = R rows of ONE batch, so B_t/C_t
// are shared by the whole CTA: an elected thread stages the [N][32*K] tiles of B and of C with
// TMA tensor copies (cp.async.bulk.tensor.2d, boxes of 128/256 timesteps x N rows, mbarrier
// complete_tx) into a 2-stage shared-memory ring; the elected thread lives in a dedicated
// producer warp; consumers release a stage through an "empty" mbarrier (one arrival per warp).  For each state n (outer loop, NU states per
// iteration for ILP) a lane
//   A3  discretises      a_k = ex2(delta_k * A2[n]),  u_k = (delta_k x_k) * B_k[n]   (smem)
//   A4  composes its K pairs in registers (P via one ex2 of A2[n]*sum(delta))
//   A5  combines across the warp with a Kogge–Stone __shfl_up_sync pair scan
//   A7  takes the carry h_in[n] of the previous tile (register, CTA-loop style)
//   A8  rescans its K steps from the exclusive prefix (a_k, u_k still in registers)
//   A9  accumulates y_k += C_k[n] * h_k (smem) ; h itself is never stored.
// x/delta/y move with coalesced 128-bit global accesses (lane owns K contiguous elements).
#pragma once

#include "selective_scan_lane_row.cuh"  // mbarrier / TMA helpers

namespace affinescan {

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
    static constexpr int kBytes = kStages * kStageBytes + 64;   // + full[2], empty[2]
    static_assert(kTileT % kBoxT == 0 && kBoxT <= 256, "tile is a whole number of boxes");
    // Bank conflicts: lane l reads the 16-byte chunks l*NV + v (v < NV) of a row.  Box and row
    // strides are multiples of 128 B, so the 8 lanes of an LDS.128 phase hit distinct 16-byte
    // slots iff NV is odd (K = 12 for fp32 io, 24 for bf16 io).
    static_assert((K * sizeof(T) / 16) % 2 == 1, "odd number of 128-bit vectors per lane");
    static_assert((kBoxT * sizeof(T)) % 128 == 0, "row stride multiple of 128 B");
};

// Non-suspending poll (mbarrier.test_wait) for the short producer-side wait.
__device__ __forceinline__ void mbar_poll(uint64_t* bar, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// NU = states processed together per n-iteration, RW = rows per warp: NU*RW independent chains
// per warp; the RW rows of a warp share every LDS of B_t/C_t (half the shared-memory traffic
// per state-step at RW = 2).
template <typename T, int VEC, int NV, int NU, int RW>
__global__ void __launch_bounds__(RW == 1 ? 384 : 256, 1)
selective_scan_warp_row_tma_kernel(const T* __restrict__ x, const T* __restrict__ delta,
                                   const float* __restrict__ A,
                                   const __grid_constant__ CUtensorMap mapB,
                                   const __grid_constant__ CUtensorMap mapC,
                                   const float* __restrict__ D, const float* __restrict__ h0,
                                   T* __restrict__ y, float* __restrict__ h_last, int batch,
                                   int d_inner, int ctas_per_batch, long long L)
{
    constexpr int K = NV * VEC;
    using S = WarpRowTmaSmem<T, K>;
    constexpr int N = S::N;
    using AccS = Access<T, VEC, true>;  // streamed once: x, delta, y

    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + S::kStages * S::kStageBytes);
    uint64_t* empty = full + S::kStages;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int R = (blockDim.x >> 5) - 1;  // consumer warps per CTA; warp R is the producer
    const int b = blockIdx.x / ctas_per_batch;
    const int d0 = (blockIdx.x - b * ctas_per_batch) * R * RW;
    bool active[RW];   // inactive rows are computed (on a valid row) but never stored: their
    int dd[RW];        // warps still take part in the stage ring
    long long row[RW];
#pragma unroll
    for (int r = 0; r < RW; ++r) {
        const int d = d0 + warp * RW + r;
        active[r] = d < d_inner;
        dd[r] = active[r] ? d : d_inner - 1;
        row[r] = static_cast<long long>(b) * d_inner + dd[r];
    }

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
    auto issue_tile = [&](long long tile) {  // one thread
        const int st = static_cast<int>(tile % S::kStages);
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
    // as every consumer warp has released it, and never touches the data itself.
    if (warp == R) {
        if (lane == 0) {
            for (long long tile = 0; tile < ntiles; ++tile) {
                if (tile >= S::kStages) {
                    const long long prev = tile - S::kStages;  // the tile that used this stage
                    mbar_poll(&empty[prev % S::kStages],
                              static_cast<unsigned>((prev / S::kStages) & 1));
                    fence_proxy_async_smem();
                }
                issue_tile(tile);
            }
        }
        return;
    }

    // Lane n keeps A2[n] = A[d,n]*log2(e) and the carry h_in[n] of each row; broadcast by shuffle.
    float A2r[RW], hcr[RW], Dd[RW];
#pragma unroll
    for (int r = 0; r < RW; ++r) {
        A2r[r] = lane < N ? __ldg(A + static_cast<long long>(dd[r]) * N + lane) * kLog2e : 0.0f;
        hcr[r] = (lane < N && h0) ? __ldg(h0 + row[r] * N + lane) : 0.0f;
        Dd[r] = D ? __ldg(D + dd[r]) : 0.0f;
    }

    // byte offset (inside a tensor's stage, state n = 0) of this lane's v-th 128-bit vector
    int voff[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const int t = lane * K + v * VEC;  // timestep inside the tile
        voff[v] = (t / S::kBoxT) * S::kBoxBytes + (t % S::kBoxT) * static_cast<int>(sizeof(T));
    }

    // A1: raw 128-bit prefetch of the lane's K timesteps of x and delta, one tile ahead
    uint4 xq[RW][NV], dq[RW][NV];
    auto prefetch = [&](long long tile) {
        const long long tl = tile * S::kTileT + lane * K;
#pragma unroll
        for (int r = 0; r < RW; ++r) {
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                xq[r][v] = make_uint4(0, 0, 0, 0);  // identity padding: delta = 0 => a = 1, u = 0
                dq[r][v] = make_uint4(0, 0, 0, 0);  // (Q12)
                if (tl + v * VEC < L) {
                    xq[r][v] = __ldcs(reinterpret_cast<const uint4*>(x + row[r] * L + tl + v * VEC));
                    dq[r][v] =
                        __ldcs(reinterpret_cast<const uint4*>(delta + row[r] * L + tl + v * VEC));
                }
            }
        }
    };
    prefetch(0);

    for (long long tile = 0; tile < ntiles; ++tile) {
        const int st = static_cast<int>(tile % S::kStages);
        const unsigned parity = static_cast<unsigned>((tile / S::kStages) & 1);
        const long long tl = tile * S::kTileT + lane * K;  // first timestep of this lane
        float dl[RW][K], dx[RW][K], yv[RW][K], dsum[RW];
#pragma unroll
        for (int r = 0; r < RW; ++r) {
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                float xv[VEC], dv[VEC];
                unpack128<T>(xq[r][v], xv);
                unpack128<T>(dq[r][v], dv);
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    dl[r][v * VEC + k] = dv[k];
                    dx[r][v * VEC + k] = dv[k] * xv[k];
                    yv[r][v * VEC + k] = Dd[r] * xv[k];
                }
            }
            dsum[r] = 0.0f;
#pragma unroll
            for (int k = 0; k < K; ++k) dsum[r] += dl[r][k];
        }
        if (tile + 1 < ntiles) prefetch(tile + 1);

        mbar_wait(&full[st], parity);
        const unsigned char* sB = smem_raw + st * S::kStageBytes;
        const unsigned char* sC = sB + S::kBoxes * S::kBoxBytes;

#pragma unroll 1
        for (int n0 = 0; n0 < N; n0 += NU) {
            float a[NU][RW][K], u[NU][RW][K];
            Pair inc[NU][RW];
            float hin[NU][RW];
            // ---- A3 + A4 for NU states x RW rows: independent work, issued back to back
#pragma unroll
            for (int j = 0; j < NU; ++j) {
                const int n = n0 + j;
                float A2n[RW];
#pragma unroll
                for (int r = 0; r < RW; ++r) {
                    A2n[r] = __shfl_sync(kFullMask, A2r[r], n);
                    hin[j][r] = __shfl_sync(kFullMask, hcr[r], n);
                }
                const unsigned char* bn = sB + n * S::kBoxT * static_cast<int>(sizeof(T));
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    float bv[VEC];  // one LDS.128 of B serves all RW rows
                    unpack128<T>(*reinterpret_cast<const uint4*>(bn + voff[v]), bv);
#pragma unroll
                    for (int r = 0; r < RW; ++r) {
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            a[j][r][v * VEC + k] = ex2_approx(dl[r][v * VEC + k] * A2n[r]);
                            u[j][r][v * VEC + k] = dx[r][v * VEC + k] * bv[k];
                        }
                    }
                }
#pragma unroll
                for (int r = 0; r < RW; ++r)
                    inc[j][r] = Pair{ex2_approx(dsum[r] * A2n[r]), u[j][r][0]};
            }
#pragma unroll
            for (int k = 1; k < K; ++k) {
#pragma unroll
                for (int j = 0; j < NU; ++j) {
#pragma unroll
                    for (int r = 0; r < RW; ++r)
                        inc[j][r].U = fmaf(a[j][r][k], inc[j][r].U, u[j][r][k]);
                }
            }
            // ---- A5: warp combine (NU*RW interleaved Kogge–Stone scans)
#pragma unroll
            for (int dlt = 1; dlt < 32; dlt <<= 1) {
                Pair pv[NU][RW];
#pragma unroll
                for (int j = 0; j < NU; ++j) {
#pragma unroll
                    for (int r = 0; r < RW; ++r) pv[j][r] = shfl_up_pair(inc[j][r], dlt);
                }
                if (lane >= dlt) {
#pragma unroll
                    for (int j = 0; j < NU; ++j) {
#pragma unroll
                        for (int r = 0; r < RW; ++r) inc[j][r] = compose(inc[j][r], pv[j][r]);
                    }
                }
            }
            // ---- A7/A8: carry-in, rescan; A9: y accumulation
#pragma unroll
            for (int j = 0; j < NU; ++j) {
                const int n = n0 + j;
                float hv[RW];
#pragma unroll
                for (int r = 0; r < RW; ++r) {
                    Pair ex = shfl_up_pair(inc[j][r], 1);
                    if (lane == 0) ex = identity_pair();
                    const Pair tot = shfl_pair(inc[j][r], 31);
                    hv[r] = apply(ex, hin[j][r]);
                    const float hout = apply(tot, hin[j][r]);  // state after the tile (uniform)
                    if (lane == n) hcr[r] = hout;
                }
                const unsigned char* cn = sC + n * S::kBoxT * static_cast<int>(sizeof(T));
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    float cc[VEC];  // one LDS.128 of C serves all RW rows
                    unpack128<T>(*reinterpret_cast<const uint4*>(cn + voff[v]), cc);
#pragma unroll
                    for (int r = 0; r < RW; ++r) {
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            hv[r] = fmaf(a[j][r][v * VEC + k], hv[r], u[j][r][v * VEC + k]);
                            yv[r][v * VEC + k] = fmaf(cc[k], hv[r], yv[r][v * VEC + k]);
                        }
                    }
                }
            }
        }
        // release the stage; the producer warp refills it with tile + 2 once every warp has
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
        // ---- A9: store y
#pragma unroll
        for (int r = 0; r < RW; ++r) {
            if (active[r]) {
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    if (tl + v * VEC < L) {
                        float out[VEC];
#pragma unroll
                        for (int k = 0; k < VEC; ++k) out[k] = yv[r][v * VEC + k];
                        AccS::store(y + row[r] * L + tl + v * VEC, out);
                    }
                }
            }
        }
    }
    // ---- A10: final state
#pragma unroll
    for (int r = 0; r < RW; ++r) {
        if (h_last && active[r] && lane < N) h_last[row[r] * N + lane] = hcr[r];
    }
}

}  // namespace affinescan
