// affinescan_affine.cu — host launch layer of affine_scan (include/affinescan.h): picks a
// kernel variant from the shape and enqueues it on the caller's stream.
#include <limits>

#include "affine_scan.cuh"
#include "host_internal.h"

namespace affinescan_host {

using namespace affinescan;
using bf16 = __nv_bfloat16;

namespace {

constexpr int kAffJ = 4;              // 128-bit vectors per thread per tile
constexpr int kAffWarps = 8;          // 256 threads
constexpr int kAffLookbackWarps = 8;  // (16 warps = 8192-element tiles measured the same on long
                                      // L, slower on short L)
constexpr int kAffLookbackJ = 4;      // look-back tiles of 4096 elements (J = 8: 202 registers)
constexpr int64_t kAffCtaLoopMinL = 8192;  // at least two CTA tiles per sequence
constexpr int kScratchSlotLookback = 0;

template <typename T, int VEC>
int launch_affine_lookback(const T* a, const T* u, const float* h0, T* h, float* h_last,
                           int64_t num_seq, int64_t L, cudaStream_t stream)
{
    // four 128-bit vectors of a and of u per thread: tiles of 4096 (fp32) / 8192 (bf16) elements;
    // the scalar-access fallback keeps 4096-element tiles
    constexpr int kJ = kAffLookbackJ;
    constexpr int kTile = kAffLookbackWarps * 32 * VEC * kJ;
    const int64_t total = num_seq * L;
    const int64_t ntiles = (total + kTile - 1) / kTile;
    if (ntiles > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    // [LookbackCtrl | ntiles descriptors]; zero-filled when fresh, never cleared afterwards
    // (epoch-tagged statuses: affine_scan.cuh)
    Scratch sc;
    AS_TRY(scratch_acquire(stream, kScratchSlotLookback,
                           sizeof(LookbackCtrl) + static_cast<size_t>(ntiles) * 16, &sc));
    auto* ctrl = static_cast<LookbackCtrl*>(sc.ptr);
    auto* desc = reinterpret_cast<unsigned long long*>(ctrl + 1);
    if constexpr (VEC > 1) {
        // vector path: persistent CTAs, a/u tiles streamed through a TMA ring (affine_scan.cuh);
        // 3 stages of 32 KB, two CTAs per SM
        constexpr int kStages = 3;
        constexpr int kCtasPerSm = 2;
        using S = ChainSmem<T, VEC, kJ, kAffLookbackWarps, kStages>;
        auto kern = affine_scan_chain_kernel<T, VEC, kJ, kAffLookbackWarps, kStages, kCtasPerSm>;
        AS_TRY(allow_dynamic_smem(reinterpret_cast<const void*>(kern), S::kBytes));
        int sms = 0;
        AS_TRY(sm_count(&sms));
        const int64_t resident = static_cast<int64_t>(sms) * kCtasPerSm;
        const unsigned grid = static_cast<unsigned>(ntiles < resident ? ntiles : resident);
        kern<<<grid, (kAffLookbackWarps + 1) * 32, S::kBytes, stream>>>(
            a, u, h0, h, h_last, total, L, ntiles, desc, ctrl);
    } else {
        affine_scan_lookback_kernel<T, VEC, kJ, kAffLookbackWarps>
            <<<static_cast<unsigned>(ntiles), kAffLookbackWarps * 32, 0, stream>>>(
                a, u, h0, h, h_last, total, L, desc, ctrl);
    }
    const int st = after_launch();
    const int st2 = scratch_release(stream, sc);
    return st != AFFINESCAN_OK ? st : st2;
}

template <typename T, int VEC>
int launch_affine_cta_loop(const T* a, const T* u, const float* h0, T* h, float* h_last,
                           int64_t num_seq, int64_t L, cudaStream_t stream)
{
    const unsigned grid = static_cast<unsigned>(num_seq < 0x7fffffffLL ? num_seq : 0x7fffffffLL);
    // short sequences: one warp per CTA keeps every lane busy; long ones: 8 warps per tile
    if (L <= static_cast<int64_t>(32 * VEC * kAffJ) * 2) {
        affine_scan_cta_loop_kernel<T, VEC, kAffJ, 1><<<grid, 32, 0, stream>>>(a, u, h0, h, h_last,
                                                                                num_seq, L);
    } else {
        affine_scan_cta_loop_kernel<T, VEC, kAffJ, kAffWarps>
            <<<grid, kAffWarps * 32, 0, stream>>>(a, u, h0, h, h_last, num_seq, L);
    }
    return after_launch();
}

template <typename T, int VEC>
int launch_affine_warp_seq(const T* a, const T* u, const float* h0, T* h, float* h_last,
                           int64_t num_seq, int64_t L, cudaStream_t stream)
{
    const int64_t blocks = (num_seq + kAffWarps - 1) / kAffWarps;
    const unsigned grid = static_cast<unsigned>(blocks < 0x7fffffffLL ? blocks : 0x7fffffffLL);
    affine_scan_warp_seq_kernel<T, VEC, kAffJ, kAffWarps>
        <<<grid, kAffWarps * 32, 0, stream>>>(a, u, h0, h, h_last, num_seq, L);
    return after_launch();
}

template <typename T>
int launch_affine_blelloch(const T* a, const T* u, const float* h0, T* h, float* h_last,
                           int64_t num_seq, int64_t L, cudaStream_t stream)
{
    const unsigned grid = static_cast<unsigned>(num_seq < 0x7fffffffLL ? num_seq : 0x7fffffffLL);
    affine_scan_blelloch_kernel<T, 512><<<grid, 512, 0, stream>>>(a, u, h0, h, h_last, num_seq, L);
    return after_launch();
}

template <typename T>
int affine_dispatch(const void* a_, const void* u_, const float* h0, void* h_, float* h_last,
                    int64_t num_seq, int64_t L, int variant, cudaStream_t stream)
{
    const T* a = static_cast<const T*>(a_);
    const T* u = static_cast<const T*>(u_);
    T* h = static_cast<T*>(h_);
    constexpr int kVec = Io<T>::kVec;
    const bool vec_ok = (L % kVec == 0) && aligned16(a) && aligned16(u) && aligned16(h);
    // AUTO: enough sequences to fill the machine with independent warps or
    // CTAs => carry in a register; otherwise split the flattened stream over tiles with the
    // decoupled look-back carry.  Thresholds scale with the SM count of the device.
    if (variant == AFFINESCAN_VARIANT_AUTO) {
        // DESIGN.md §6.6, from the r02 sweeps (2^20 .. 2^30 elements, S = 1 .. 2^22, both dtypes).
        // The persistent look-back stream costs the same whatever the segmentation once a tile
        // lies inside a sequence; one CTA (or warp) per sequence wins a few percent when there are
        // several waves of sequences of moderate length; very short sequences leave most lanes of
        // a per-sequence warp idle, so the flattened stream wins again.
        int sms = 0;
        AS_TRY(sm_count(&sms));
        const bool narrow = sizeof(T) == 2;
        const int64_t waves16 = static_cast<int64_t>(sms) * 16;  // four waves of 4 CTAs per SM
        // sequences that divide the look-back tile take its aligned path (no carry, flags computed
        // once per thread): as fast as interior tiles
        const int64_t lb_tile = kAffLookbackWarps * 32 * kVec * kAffLookbackJ;
        const bool aligned = vec_ok && L < lb_tile && lb_tile % L == 0;
        const bool tiny = num_seq * L < (1 << 16);
        if (narrow) {
            if (L >= 16384 || ((aligned || L <= 512) && !tiny)) variant = AFFINESCAN_AFFINE_LOOKBACK;
            else if (L <= 2048) variant = AFFINESCAN_AFFINE_CTA_LOOP;  // one warp per sequence
            else
                variant = num_seq >= static_cast<int64_t>(sms) * 8 ? AFFINESCAN_AFFINE_WARP_SEQ
                          : L <= kAffCtaLoopMinL                   ? AFFINESCAN_AFFINE_CTA_LOOP
                                                                   : AFFINESCAN_AFFINE_LOOKBACK;
        } else {
            if (L <= 256) variant = tiny ? AFFINESCAN_AFFINE_CTA_LOOP : AFFINESCAN_AFFINE_LOOKBACK;
            else if (L <= 1024) variant = AFFINESCAN_AFFINE_CTA_LOOP;  // one warp per sequence
            else if (L < 4096)
                variant = (aligned && !tiny) ? AFFINESCAN_AFFINE_LOOKBACK : AFFINESCAN_AFFINE_CTA_LOOP;
            else
                // r03: no upper bound on L here: with >= four waves of sequences the CTA loop
                // beats the look-back stream at L = 2^17 / 2^18 too (2^30 elements: 1.89 / 1.93
                // against 2.09 / 2.15 ms)
                variant = num_seq >= waves16 ? AFFINESCAN_AFFINE_CTA_LOOP
                          : L <= kAffCtaLoopMinL                ? AFFINESCAN_AFFINE_CTA_LOOP
                                                                : AFFINESCAN_AFFINE_LOOKBACK;
        }
        // AFFINESCAN_OPT_DETERMINISTIC: the look-back folds whichever aggregates are published
        // when it polls; the register-carry schedules have one fixed association order
        if (variant == AFFINESCAN_AFFINE_LOOKBACK && deterministic_auto())
            variant = AFFINESCAN_AFFINE_CTA_LOOP;
    }
    int st;
    switch (variant) {
    case AFFINESCAN_AFFINE_WARP_SEQ:
        st = vec_ok ? launch_affine_warp_seq<T, kVec>(a, u, h0, h, h_last, num_seq, L, stream)
                    : launch_affine_warp_seq<T, 1>(a, u, h0, h, h_last, num_seq, L, stream);
        break;
    case AFFINESCAN_AFFINE_LOOKBACK:
        st = vec_ok ? launch_affine_lookback<T, kVec>(a, u, h0, h, h_last, num_seq, L, stream)
                    : launch_affine_lookback<T, 1>(a, u, h0, h, h_last, num_seq, L, stream);
        break;
    case AFFINESCAN_AFFINE_CTA_LOOP:
        st = vec_ok ? launch_affine_cta_loop<T, kVec>(a, u, h0, h, h_last, num_seq, L, stream)
                    : launch_affine_cta_loop<T, 1>(a, u, h0, h, h_last, num_seq, L, stream);
        break;
    case AFFINESCAN_AFFINE_BLELLOCH:
        st = launch_affine_blelloch<T>(a, u, h0, h, h_last, num_seq, L, stream);
        break;
    default:
        return AFFINESCAN_ERR_UNSUPPORTED;
    }
    if (st == AFFINESCAN_OK) set_last_variant(variant);
    return st;
}

__global__ void fill_h_last_kernel(const float* __restrict__ h0, float* __restrict__ h_last,
                                   long long n)
{
    const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < n) h_last[i] = h0 ? h0[i] : 0.0f;
}

}  // namespace

int fill_h_last(const float* h0, float* h_last, int64_t n, cudaStream_t stream)
{
    if (!h_last || n <= 0) return AFFINESCAN_OK;
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    fill_h_last_kernel<<<static_cast<unsigned>(blocks), 256, 0, stream>>>(h0, h_last, n);
    return after_launch();
}

int affine_scan_impl(const void* a, const void* u, const float* h0, void* h, float* h_last,
                     int64_t num_seq, int64_t L, int io_dtype, int variant, void* cuda_stream)
{
    set_last_variant(0);
    if (io_dtype != AFFINESCAN_F32 && io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (num_seq < 0 || L < 0) return AFFINESCAN_ERR_SHAPE;
    int64_t total = 0;
    if (mul_overflows(num_seq, L, &total) || total > (std::numeric_limits<int64_t>::max() >> 3))
        return AFFINESCAN_ERR_SHAPE;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (num_seq == 0) return AFFINESCAN_OK;
    if (L == 0) return fill_h_last(h0, h_last, num_seq, stream);  // h_last <- h0 (or 0)
    if (!a || !u || !h) return AFFINESCAN_ERR_NULL;
    return io_dtype == AFFINESCAN_F32
               ? affine_dispatch<float>(a, u, h0, h, h_last, num_seq, L, variant, stream)
               : affine_dispatch<bf16>(a, u, h0, h, h_last, num_seq, L, variant, stream);
}

}  // namespace affinescan_host
