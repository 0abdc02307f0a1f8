// selective_scan_lane_row.cuh — variant AFFINESCAN_SELECTIVE_LANE_ROW of
// selective_scan_fwd (include/affinescan.h; BJ north_star; SURVEY §8a A1-A10, App. A "G=1").
//
// One LANE owns one (b,d) row and walks L sequentially with all N=16 states h[n] and
// A2[n] = A[d,n]*log2(e) in registers: no shuffle, no rescan, no cross-lane reduction —
// per state-step exactly 1 MUFU.EX2 + 4 FP32 ops (arg, u, h-update, y-accumulate), the
// minimum the recurrence needs.  This is the schedule for many-row shapes
// (cfg3: 32768 rows), where the kernel is bound by the SFU/FP32 pipes, not by HBM.
//
// A warp = 32 consecutive d of one batch b, so B_t/C_t are warp-uniform.  Each warp
// stages its [2][N][TC] B/C tile with TMA bulk copies (cp.async.bulk + mbarrier
// complete_tx, double-buffered), transposes/widens it once to an fp32 [TC][2][N] tile,
// and then every state-step reads B/C with broadcast LDS.128 (one request serves 4 n for
// all 32 lanes).  x/delta come from global memory one 128-bit group ahead (register
// prefetch); y leaves with one 128-bit store per group.  Warps are autonomous: no CTA
// barrier anywhere.
#pragma once

#include "common.cuh"

namespace affinescan {

__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, unsigned parity)
{
    unsigned ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
// TMA 1-D bulk copy global -> shared, completion reported to an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void tma_bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes,
                                             uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

template <typename T, int TC>
struct LaneRowSmem {
    static constexpr int N = 16;
    static constexpr int kRawPitch = TC * static_cast<int>(sizeof(T)) + 16;  // bytes; ≡16 mod 128
    static constexpr int kRawStage = 2 * N * kRawPitch;                      // B rows then C rows
    static constexpr int kBcTile = TC * 2 * N * 4;                           // fp32 [TC][2][N]
    static constexpr int kPerWarp = 2 * kRawStage + kBcTile + 16;            // + 2 mbarriers
};

template <typename T, int TC, int WARPS>
__global__ void __launch_bounds__(WARPS * 32)
selective_scan_lane_row_kernel(const T* __restrict__ x, const T* __restrict__ delta,
                               const float* __restrict__ A, const T* __restrict__ B,
                               const T* __restrict__ C, const float* __restrict__ D,
                               const float* __restrict__ h0, T* __restrict__ y,
                               float* __restrict__ h_last, int batch, int d_inner, long long L)
{
    using S = LaneRowSmem<T, TC>;
    constexpr int N = S::N;
    constexpr int VEC = Io<T>::kVec;          // timesteps per 128-bit access
    constexpr int kChunks = TC / VEC;         // 128-bit chunks per raw row
    using Acc = Access<T, VEC, true>;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const long long rows = static_cast<long long>(batch) * d_inner;
    const long long row0 = (static_cast<long long>(blockIdx.x) * WARPS + warp) * 32;
    if (row0 >= rows) return;  // whole warp exits together; warps never sync with each other
    const long long row = row0 + lane;
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
    // lane r stages raw row r: rows 0..15 = B[b, r, :], rows 16..31 = C[b, r-16, :]
    const T* my_src = (lane < N ? B : C) + (static_cast<long long>(b) * N + (lane & (N - 1))) * L;
    auto issue_tile = [&](long long tile) {
        const int st = static_cast<int>(tile & 1);
        const long long t0 = tile * TC;
        const long long rem = L - t0;
        const unsigned row_bytes = static_cast<unsigned>((rem < TC ? rem : TC) * sizeof(T));
        if (lane == 0) mbar_arrive_expect_tx(&full[st], row_bytes * 2u * N);
        __syncwarp();
        tma_bulk_g2s(wbase + st * S::kRawStage + lane * S::kRawPitch, my_src + t0, row_bytes, &full[st]);
    };
    issue_tile(0);
    if (ntiles > 1) issue_tile(1);

    // per-row constants and state
    float A2[N], h[N];
#pragma unroll
    for (int q = 0; q < N / 4; ++q) {
        const float4 av = __ldg(reinterpret_cast<const float4*>(A + static_cast<long long>(d) * N) + q);
        A2[4 * q + 0] = av.x * kLog2e; A2[4 * q + 1] = av.y * kLog2e;
        A2[4 * q + 2] = av.z * kLog2e; A2[4 * q + 3] = av.w * kLog2e;
        float4 hv = make_float4(0.f, 0.f, 0.f, 0.f);
        if (h0) hv = __ldg(reinterpret_cast<const float4*>(h0 + row * N) + q);
        h[4 * q + 0] = hv.x; h[4 * q + 1] = hv.y; h[4 * q + 2] = hv.z; h[4 * q + 3] = hv.w;
    }
    const float Dd = D ? __ldg(D + d) : 0.0f;

    const T* xr = x + row * L;
    const T* dr = delta + row * L;
    T* yr = y + row * L;

    // A1: register prefetch, one 128-bit group (VEC timesteps) ahead
    float xn[VEC], dn[VEC];
    Acc::load(xr, xn);
    Acc::load(dr, dn);

    for (long long tile = 0; tile < ntiles; ++tile) {
        const int st = static_cast<int>(tile & 1);
        const unsigned parity = static_cast<unsigned>((tile >> 1) & 1);
        const long long t0 = tile * TC;
        mbar_wait(&full[st], parity);
        __syncwarp();  // every lane is done reading the fp32 tile of the previous iteration
        // A2: widen + transpose raw [2N][TC] (io dtype) -> bc [TC][2][N] (fp32).
        // Raw pitch ≡ 16 (mod 128) bytes makes the LDS.128 conflict-free across rows; the
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

        // A3..A9: sequential in t, all N states in registers
        for (int g = 0; g < kChunks; ++g) {
            const long long tg = t0 + g * VEC;
            if (tg >= L) break;  // warp-uniform
            float xv[VEC], dl[VEC];
#pragma unroll
            for (int k = 0; k < VEC; ++k) { xv[k] = xn[k]; dl[k] = dn[k]; }
            if (tg + VEC < L) {
                Acc::load(xr + tg + VEC, xn);
                Acc::load(dr + tg + VEC, dn);
            }
            float out[VEC];
#pragma unroll
            for (int k = 0; k < VEC; ++k) {
                const float dlk = dl[k];
                const float dxk = dlk * xv[k];
                float acc0 = Dd * xv[k], acc1 = 0.0f;
                const float4* bc4 = reinterpret_cast<const float4*>(bc + (g * VEC + k) * 2 * N);
#pragma unroll
                for (int q = 0; q < N / 4; ++q) {
                    const float4 b4 = bc4[q];
                    const float4 c4 = bc4[N / 4 + q];
                    h[4 * q + 0] = fmaf(ex2_approx(dlk * A2[4 * q + 0]), h[4 * q + 0], dxk * b4.x);
                    acc0 = fmaf(c4.x, h[4 * q + 0], acc0);
                    h[4 * q + 1] = fmaf(ex2_approx(dlk * A2[4 * q + 1]), h[4 * q + 1], dxk * b4.y);
                    acc1 = fmaf(c4.y, h[4 * q + 1], acc1);
                    h[4 * q + 2] = fmaf(ex2_approx(dlk * A2[4 * q + 2]), h[4 * q + 2], dxk * b4.z);
                    acc0 = fmaf(c4.z, h[4 * q + 2], acc0);
                    h[4 * q + 3] = fmaf(ex2_approx(dlk * A2[4 * q + 3]), h[4 * q + 3], dxk * b4.w);
                    acc1 = fmaf(c4.w, h[4 * q + 3], acc1);
                }
                out[k] = acc0 + acc1;
            }
            Acc::store(yr + tg, out);
        }
    }
    // A10: final state
    if (h_last) {
#pragma unroll
        for (int q = 0; q < N / 4; ++q)
            reinterpret_cast<float4*>(h_last + row * N)[q] =
                make_float4(h[4 * q + 0], h[4 * q + 1], h[4 * q + 2], h[4 * q + 3]);
    }
}

}  // namespace affinescan
