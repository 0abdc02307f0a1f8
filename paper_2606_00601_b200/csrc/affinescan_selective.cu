// affinescan_selective.cu — host launch layer of selective_scan_fwd and its extended forms
// (include/affinescan.h): validates, picks a kernel variant from the shape, encodes (and caches)
// the TMA tensor maps of B and C, and enqueues ONE kernel on the caller's stream.
#include <atomic>
#include <limits>
#include <map>
#include <mutex>
#include <tuple>

#include "host_internal.h"
#include "selective_scan_lane_row.cuh"
#include "selective_scan_warp_row.cuh"
#include "selective_scan_warp_row_tma.cuh"

namespace affinescan_host {

using namespace affinescan;
using bf16 = __nv_bfloat16;

namespace {

constexpr int kWarpRowTmaMaxWarps = 11;   // warp_row_tma: rows per CTA (+1 producer warp = 384 threads)
constexpr int64_t kWarpRowTmaMinL = 1024; // below two warp tiles the plain warp_row is as good
constexpr int64_t kChunkedMinL = 8192;    // chunked (look-back) schedule: at least ~10 tiles per row
constexpr int kSelWarps = 4;        // warp_row: rows per CTA
#ifndef LR_TC
#define LR_TC 32
#endif
constexpr int kLaneRowTc = LR_TC;   // lane_row: timesteps per staged B/C tile
constexpr int kLaneRowWarps = 4;    // lane_row: warps per CTA (autonomous)
constexpr int kLaneRowDefaultPoly16 = 4;  // sixteenths of the exps done on the fma pipe

// Tuning knobs of the lane_row schedule (affinescan_set_option); -1 = choose from the shape.
std::atomic<int> g_opt_lane_row_g{-1};
std::atomic<int> g_opt_lane_row_poly16{-1};

// ---------------------------------------------------------------- TMA tensor maps
// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda).
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                   const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                   const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int get_encode_tiled(EncodeTiledFn* out)
{
    static std::atomic<void*> cached{nullptr};
    void* fn = cached.load(std::memory_order_acquire);
    if (!fn) {
        cudaDriverEntryPointQueryResult qres;
        AS_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (qres != cudaDriverEntryPointSuccess || !fn) return cuda_fail(cudaErrorNotSupported);
        cached.store(fn, std::memory_order_release);
    }
    *out = reinterpret_cast<EncodeTiledFn>(fn);
    return AFFINESCAN_OK;
}

// Tensor map over a [rows = batch*N, L] io-dtype matrix (B or C), box = {box_t timesteps, N rows}.
// A map depends only on (pointer, shape, box, dtype), so it is encoded once and cached: repeated
// calls on the same tensors (a training loop, a replayed graph) pay a map lookup, not a driver
// call.  The cache is bounded; it is dropped when full.
struct MapKey {
    const void* base;
    int64_t rows, L;
    int box_t, N, esize, swizzle;
    bool operator<(const MapKey& o) const
    {
        return std::tie(base, rows, L, box_t, N, esize, swizzle) <
               std::tie(o.base, o.rows, o.L, o.box_t, o.N, o.esize, o.swizzle);
    }
};
std::mutex g_map_mu;
std::map<MapKey, CUtensorMap> g_maps;
constexpr size_t kMaxCachedMaps = 512;

// swizzle128 = the 128-byte shared-memory swizzle (box rows of exactly 128 B: the x / delta rings)
template <typename T>
int make_bc_tensor_map(CUtensorMap* map, const T* base, int64_t rows, int64_t L, int box_t, int N,
                       bool swizzle128 = false)
{
    const MapKey key{base, rows, L, box_t, N, static_cast<int>(sizeof(T)), swizzle128 ? 1 : 0};
    {
        std::lock_guard<std::mutex> lk(g_map_mu);
        auto it = g_maps.find(key);
        if (it != g_maps.end()) {
            *map = it->second;
            return AFFINESCAN_OK;
        }
    }
    EncodeTiledFn encode = nullptr;
    AS_TRY(get_encode_tiled(&encode));
    const cuuint64_t dims[2] = {static_cast<cuuint64_t>(L), static_cast<cuuint64_t>(rows)};
    const cuuint64_t strides[1] = {static_cast<cuuint64_t>(L) * sizeof(T)};
    const cuuint32_t box[2] = {static_cast<cuuint32_t>(box_t), static_cast<cuuint32_t>(N)};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode(map, sizeof(T) == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                                  : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                              2, const_cast<T*>(base), dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE,
                              swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cuda_fail(cudaErrorInvalidValue);
    std::lock_guard<std::mutex> lk(g_map_mu);
    if (g_maps.size() >= kMaxCachedMaps) g_maps.clear();
    g_maps[key] = *map;
    return AFFINESCAN_OK;
}

template <typename Kern>
int allow_smem(Kern kern, int bytes)
{
    return allow_dynamic_smem(reinterpret_cast<const void*>(kern), bytes);
}

// ---------------------------------------------------------------- typed view of the arguments
template <typename T>
struct Typed {
    const T *x, *delta, *B, *C;
    T* y;
    const float *A, *D, *h0;
    float* h_last;
    SelectiveExt ext;
    bool has_ext;
    int batch, d_inner, N;
    int64_t L;
};

template <typename T>
Typed<T> typed(const SelectiveArgs& a)
{
    Typed<T> t;
    t.x = static_cast<const T*>(a.x);
    t.delta = static_cast<const T*>(a.delta);
    t.B = static_cast<const T*>(a.B);
    t.C = static_cast<const T*>(a.C);
    t.y = static_cast<T*>(a.y);
    t.A = a.A;
    t.D = a.D;
    t.h0 = a.h0;
    t.h_last = a.h_last;
    t.ext = SelectiveExt{a.z, a.delta_bias, a.reset, a.delta_softplus};
    t.has_ext = a.z || a.delta_bias || a.reset || a.delta_softplus;
    t.batch = a.batch;
    t.d_inner = a.d_inner;
    t.N = a.N;
    t.L = a.L;
    return t;
}

// ---------------------------------------------------------------- warp_row (general fallback)
template <typename T, int VEC, int NV, bool EXT>
int launch_warp_row_inst(const Typed<T>& t, cudaStream_t stream)
{
    const int64_t rows = static_cast<int64_t>(t.batch) * t.d_inner;
    const int64_t blocks = (rows + kSelWarps - 1) / kSelWarps;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    selective_scan_warp_row_kernel<T, VEC, NV, kSelWarps, EXT>
        <<<static_cast<unsigned>(blocks), kSelWarps * 32, 0, stream>>>(
            t.x, t.delta, t.A, t.B, t.C, t.D, t.h0, t.y, t.h_last, t.ext, t.batch, t.d_inner, t.N,
            t.L);
    return after_launch();
}

template <typename T>
int launch_warp_row(const Typed<T>& t, bool vec_ok, cudaStream_t stream)
{
    constexpr int kVec = Io<T>::kVec;
    if (vec_ok)
        return t.has_ext ? launch_warp_row_inst<T, kVec, 16 / kVec, true>(t, stream)
                         : launch_warp_row_inst<T, kVec, 16 / kVec, false>(t, stream);
    return t.has_ext ? launch_warp_row_inst<T, 1, 4, true>(t, stream)
                     : launch_warp_row_inst<T, 1, 4, false>(t, stream);
}

// ---------------------------------------------------------------- lane_row (many rows)
template <typename T, int G, int F16, int EXT, int ASTR, int ORDER = 0, int WARPS = kLaneRowWarps>
int launch_lane_row_inst(const Typed<T>& t, cudaStream_t stream)
{
    // polynomial degree per io dtype: DESIGN.md §7 (tolerance argument)
    constexpr int kDeg = sizeof(T) == 2 ? 3 : 5;
    using S = LaneRowSmem<T, kLaneRowTc>;
    auto kern = selective_scan_lane_row_kernel<T, G, kLaneRowTc, WARPS, F16, kDeg, EXT, ASTR, ORDER>;
    constexpr int smem = S::kPerWarp * WARPS;
    AS_TRY(allow_smem(kern, smem));
    CUtensorMap mapB, mapC;
    AS_TRY(make_bc_tensor_map<T>(&mapB, t.B, static_cast<int64_t>(t.batch) * 16, t.L, kLaneRowTc, 16));
    AS_TRY(make_bc_tensor_map<T>(&mapC, t.C, static_cast<int64_t>(t.batch) * 16, t.L, kLaneRowTc, 16));
    const int64_t rows = static_cast<int64_t>(t.batch) * t.d_inner;
    const int64_t warps = rows / (32 / G);
    const int64_t blocks = (warps + WARPS - 1) / WARPS;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    kern<<<static_cast<unsigned>(blocks), WARPS * 32, smem, stream>>>(
        t.x, t.delta, t.A, mapB, mapC, t.D, t.h0, t.y, t.h_last, t.ext, t.batch, t.d_inner, t.L);
    return after_launch();
}

// Composition of the balanced grid for `rows` rows: the rows are cut into the fewest rounds of at
// most 224 rows per SM, and a round gives every sub-partition u units of 8 rows (u <= 7) as q2
// two-lane warps (2 units) and q4 four-lane warps (1 unit).
// Returns the number of rounds.
int64_t lane_mix_shape(int64_t rows, int sms, int* q2, int* q4, int* units = nullptr)
{
    const int64_t cap = static_cast<int64_t>(sms) * 224;
    const int64_t rounds = rows <= 0 ? 1 : (rows + cap - 1) / cap;
    const int64_t per_sm = (rows + rounds * sms - 1) / (rounds * sms);
    int u = static_cast<int>((per_sm + 31) / 32);
    u = u < 1 ? 1 : (u > 7 ? 7 : u);
    // measured best composition per u (r02 sweep): four-lane warps pay twice the per-timestep
    // work per row, but a sub-partition wants two or three warps to hide latencies
    static const int kQ2[8] = {0, 0, 0, 1, 1, 2, 3, 3};
    static const int kQ4[8] = {0, 1, 2, 1, 2, 1, 0, 1};
    *q2 = kQ2[u];
    *q4 = kQ4[u];
    if (units) *units = u;
    return rounds;
}

template <typename T, int F16, int EXT, int ORDER>
int launch_lane_mix_inst(const Typed<T>& t, cudaStream_t stream)
{
    constexpr int kDeg = sizeof(T) == 2 ? 3 : 5;
    using M = LaneMixSmem<T, kLaneRowTc>;
    auto kern = selective_scan_lane_mix_kernel<T, kLaneRowTc, F16, kDeg, EXT, ORDER>;
    constexpr int smem = M::kBytes;
    // a CTA's 224 consecutive rows must lie in at most kMixMaxBatches batches
    if (t.d_inner < 224 || t.d_inner % 32 != 0) return AFFINESCAN_ERR_UNSUPPORTED;
    AS_TRY(allow_smem(kern, smem));
    CUtensorMap mapB, mapC;
    AS_TRY(make_bc_tensor_map<T>(&mapB, t.B, static_cast<int64_t>(t.batch) * 16, t.L, kLaneRowTc, 16));
    AS_TRY(make_bc_tensor_map<T>(&mapC, t.C, static_cast<int64_t>(t.batch) * 16, t.L, kLaneRowTc, 16));
    // x and delta as [rows, L] matrices, boxes of {128 bytes, 8 rows}, 128-byte swizzle
    CUtensorMap mapX, mapD;
    const int64_t rows = static_cast<int64_t>(t.batch) * t.d_inner;
    constexpr int kBoxT = 128 / static_cast<int>(sizeof(T));
    AS_TRY(make_bc_tensor_map<T>(&mapX, t.x, rows, t.L, kBoxT, 8, true));
    AS_TRY(make_bc_tensor_map<T>(&mapD, t.delta, rows, t.L, kBoxT, 8, true));
    int sms = 0;
    AS_TRY(sm_count(&sms));
    int q2 = 0, q4 = 0;
    lane_mix_shape(rows, sms, &q2, &q4);
    kern<<<static_cast<unsigned>(sms), 16 * 32, smem, stream>>>(
        t.x, t.delta, t.A, mapB, mapC, mapX, mapD, t.D, t.h0, t.y, t.h_last, t.ext, t.batch,
        t.d_inner, t.L, q2, q4);
    return after_launch();
}

// the gated Mamba block (softplus + z, no resets) has a branch-free instantiation; any other
// combination of fused steps takes the generic one
template <typename T>
bool is_gated(const Typed<T>& t)
{
    return t.ext.delta_softplus && t.ext.z && !t.ext.reset;
}

template <typename T, int G, int F16>
int launch_lane_row_gf(const Typed<T>& t, cudaStream_t stream)
{
    // G = 1 (one or two warps per sub-partition): pass-major; G = 2: timestep-major
    constexpr int kOrder = G == 1 ? 0 : 1;
    if (!t.has_ext) return launch_lane_row_inst<T, G, F16, 0, 0, kOrder>(t, stream);
    if (G == 1 && is_gated(t)) return launch_lane_row_inst<T, 1, F16, kExtGated, 0, 0>(t, stream);
    return launch_lane_row_inst<T, G, F16, kExtGeneric, 0, kOrder>(t, stream);
}

// Grid of the lane_row schedule from the row count: modelled cycles per timestep
// on the busiest sub-partition, fitted to the r02 sweeps on B200 (w = row warps resident there).
// Returns the cost of the best grid; *G = 1 | 2 (lanes per row, uniform grid) | 3 (balanced grid).
int64_t lane_grid_cost(int64_t rows, int d_inner, int sms, bool wide, int* G)
{
    const int64_t smsp = static_cast<int64_t>(sms) * 4;
    const int64_t w1 = (rows / 32 + smsp - 1) / smsp, w2 = (rows / 16 + smsp - 1) / smsp;
    int q2 = 0, q4 = 0, u = 0;
    const int64_t rounds = lane_mix_shape(rows, sms, &q2, &q4, &u);
    // fp32 io pays more per warp (wider tiles, degree-5 polynomial)
    const int64_t c1 = wide ? 350 * w1 : (w1 == 1 ? 215 : 40 + 150 * w1);
    const int64_t c2 = wide ? 20 + 150 * w2 : (w2 == 1 ? 143 : 45 + 80 * w2);
    // balanced grid: cost of a round by units of 8 rows per sub-partition
    static const int kMix16[8] = {0, 126, 155, 189, 206, 236, 288, 290};
    static const int kMix32[8] = {0, 161, 189, 236, 232, 283, 338, 332};
    const int64_t c3 = d_inner >= 224 ? (wide ? kMix32[u] : kMix16[u]) * rounds
                                      : std::numeric_limits<int64_t>::max();
    *G = (c3 < c1 && c3 < c2) ? 3 : (c2 < c1 ? 2 : 1);
    return *G == 3 ? c3 : (*G == 2 ? c2 : c1);
}

template <typename T>
int launch_lane_row(const Typed<T>& t, int a_structure, cudaStream_t stream)
{
    if (a_structure == AFFINESCAN_A_SCALAR_PER_ROW)
        return t.has_ext ? launch_lane_row_inst<T, 1, 0, kExtGeneric, 1>(t, stream)
                         : launch_lane_row_inst<T, 1, 0, 0, 1>(t, stream);
    if (a_structure == AFFINESCAN_A_POWERS)
        return t.has_ext ? launch_lane_row_inst<T, 1, 0, kExtGeneric, 2>(t, stream)
                         : launch_lane_row_inst<T, 1, 0, 0, 2>(t, stream);
    int G = g_opt_lane_row_g.load(std::memory_order_relaxed);
    int poly16 = g_opt_lane_row_poly16.load(std::memory_order_relaxed);
    if (G < 0) {
        int sms = 0;
        AS_TRY(sm_count(&sms));
        lane_grid_cost(static_cast<int64_t>(t.batch) * t.d_inner, t.d_inner, sms, sizeof(T) == 4, &G);
        if (poly16 < 0) poly16 = G == 1 ? kLaneRowDefaultPoly16 : 0;
    }
    if (poly16 < 0) poly16 = kLaneRowDefaultPoly16;
    if (G == 3) {   // balanced grid: three G = 2 warps + one G = 4 warp per sub-partition
        if (t.d_inner < 224) return AFFINESCAN_ERR_UNSUPPORTED;
#ifndef LR_MIX_ORDER
#define LR_MIX_ORDER 1
#endif
        if (!t.has_ext) return launch_lane_mix_inst<T, 0, 0, LR_MIX_ORDER>(t, stream);
        if (is_gated(t)) return launch_lane_mix_inst<T, 0, kExtGated, 1>(t, stream);
        return launch_lane_mix_inst<T, 0, kExtGeneric, 1>(t, stream);
    }
    if (G == 1 && poly16 == 0) return launch_lane_row_gf<T, 1, 0>(t, stream);
    if (G == 1 && poly16 == 4) return launch_lane_row_gf<T, 1, 4>(t, stream);
    // the polynomial only pays with one or two warps per sub-partition: the
    // two-lane and balanced grids always take every 2^x on the MUFU
    if (G == 2) return launch_lane_row_gf<T, 2, 0>(t, stream);
    return AFFINESCAN_ERR_UNSUPPORTED;
}

// ---------------------------------------------------------------- warp_row_tma (few rows)
constexpr int kScratchSlotChunked = 1;

template <typename T>
struct TmaShape {
    static constexpr int kVec = Io<T>::kVec;
    // odd: conflict-free LDS.128 (K = 12 fp32 / 24 bf16 timesteps per lane; K = 20 with one
    // chain measured slower: cfg4 0.906 vs 0.818 ms)
    static constexpr int kNv = 3;
    // fp32 io: two states per n-iteration (two independent chains); bf16 io: K = 24 leaves
    // registers for one chain only.
    static constexpr int kNu = sizeof(T) == 2 ? 1 : 2;
    using S = WarpRowTmaSmem<T, kNv * kVec>;
};

// CHUNKED: persistent CTAs draw (tile, row-block) items tile-major; carry by decoupled look-back
template <typename T, bool EXT>
int launch_chunked_inst(const Typed<T>& t, cudaStream_t stream)
{
    using Sh = TmaShape<T>;
    using S = typename Sh::S;
    auto kern = selective_scan_warp_row_tma_kernel<T, Sh::kVec, Sh::kNv, Sh::kNu, EXT, true>;
    AS_TRY(allow_smem(kern, S::kBytes));
    CUtensorMap mapB, mapC;
    AS_TRY(make_bc_tensor_map<T>(&mapB, t.B, static_cast<int64_t>(t.batch) * 16, t.L, S::kBoxT, 16));
    AS_TRY(make_bc_tensor_map<T>(&mapC, t.C, static_cast<int64_t>(t.batch) * 16, t.L, S::kBoxT, 16));
    int sms = 0;
    AS_TRY(sm_count(&sms));
    // 5 row-warps + the producer warp = 192 threads: two CTAs per SM (2 x 192 x 168 registers,
    // 2 x 98 KB of staging), so one CTA's ticket + TMA latency hides behind the other's arithmetic
    constexpr int kChunkedWarps = 5;
    const int R = t.d_inner < kChunkedWarps ? t.d_inner : kChunkedWarps;
    const int ctas_per_batch = (t.d_inner + R - 1) / R;
    const int64_t ntiles = (t.L + S::kTileT - 1) / S::kTileT;
    int64_t nitems = 0, ndesc = 0;
    const int64_t rows = static_cast<int64_t>(t.batch) * t.d_inner;
    if (mul_overflows(ntiles, static_cast<int64_t>(t.batch) * ctas_per_batch, &nitems) ||
        nitems > 0x7ffffff0LL || mul_overflows(rows * 16, ntiles, &ndesc) ||
        ndesc > (std::numeric_limits<int64_t>::max() >> 5))
        return AFFINESCAN_ERR_UNSUPPORTED;
    // [LookbackCtrl | rows x ntiles x N descriptors of 16 B]; zero-filled when fresh, never
    // cleared afterwards (epoch-tagged statuses)
    Scratch sc;
    AS_TRY(scratch_acquire(stream, kScratchSlotChunked,
                           sizeof(LookbackCtrl) + static_cast<size_t>(ndesc) * 16, &sc));
    auto* ctrl = static_cast<LookbackCtrl*>(sc.ptr);
    auto* desc = reinterpret_cast<unsigned long long*>(ctrl + 1);
    const int64_t grid = nitems < 2 * sms ? nitems : 2 * sms;  // two persistent CTAs per SM
    kern<<<static_cast<unsigned>(grid), (R + 1) * 32, S::kBytes, stream>>>(
        t.x, t.delta, t.A, mapB, mapC, t.D, t.h0, t.y, t.h_last, t.ext, t.batch, t.d_inner,
        ctas_per_batch, t.L, desc, ctrl);
    const int st = after_launch();
    const int st2 = scratch_release(stream, sc);
    return st != AFFINESCAN_OK ? st : st2;
}

template <typename T>
int launch_chunked(const Typed<T>& t, cudaStream_t stream)
{
    return t.has_ext ? launch_chunked_inst<T, true>(t, stream)
                     : launch_chunked_inst<T, false>(t, stream);
}

template <typename T, bool EXT>
int launch_warp_row_tma_inst(const Typed<T>& t, cudaStream_t stream)
{
    using Sh = TmaShape<T>;
    using S = typename Sh::S;
    auto kern = selective_scan_warp_row_tma_kernel<T, Sh::kVec, Sh::kNv, Sh::kNu, EXT, false>;
    AS_TRY(allow_smem(kern, S::kBytes));
    CUtensorMap mapB, mapC;
    AS_TRY(make_bc_tensor_map<T>(&mapB, t.B, static_cast<int64_t>(t.batch) * 16, t.L, S::kBoxT, 16));
    AS_TRY(make_bc_tensor_map<T>(&mapC, t.C, static_cast<int64_t>(t.batch) * 16, t.L, S::kBoxT, 16));
    // R rows (warps) of one batch per CTA, sized so that one wave of CTAs covers all rows when
    // they fit (cfg2/cfg4 on 148 SMs: 1536 rows -> 140 CTAs of 11 warps)
    int sms = 0;
    AS_TRY(sm_count(&sms));
    const int slots = sms / t.batch > 0 ? sms / t.batch : 1;
    int R = (t.d_inner + slots - 1) / slots;  // consumer warps per CTA
    R = R < 1 ? 1 : (R > kWarpRowTmaMaxWarps ? kWarpRowTmaMaxWarps : R);
    const int ctas_per_batch = (t.d_inner + R - 1) / R;
    const int64_t blocks = static_cast<int64_t>(t.batch) * ctas_per_batch;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    kern<<<static_cast<unsigned>(blocks), (R + 1) * 32, S::kBytes, stream>>>(
        t.x, t.delta, t.A, mapB, mapC, t.D, t.h0, t.y, t.h_last, t.ext, t.batch, t.d_inner,
        ctas_per_batch, t.L, nullptr, nullptr);
    return after_launch();
}

template <typename T>
int launch_warp_row_tma(const Typed<T>& t, cudaStream_t stream)
{
    return t.has_ext ? launch_warp_row_tma_inst<T, true>(t, stream)
                     : launch_warp_row_tma_inst<T, false>(t, stream);
}

// ---------------------------------------------------------------- dispatch
template <typename T>
int selective_dispatch(const SelectiveArgs& a, cudaStream_t stream)
{
    const Typed<T> t = typed<T>(a);
    constexpr int kVec = Io<T>::kVec;
    const bool vec_ok = (t.L % kVec == 0) && aligned16(t.x) && aligned16(t.delta) &&
                        aligned16(t.B) && aligned16(t.C) && (!t.y || aligned16(t.y)) &&
                        (!a.z || aligned16(a.z));
    const bool lane_ok_common = vec_ok && t.L < (1LL << 31) - 4096;  // TMA coordinates are int32
    const bool lane_ok = lane_ok_common && t.N == 16 && (t.d_inner % 32 == 0) && aligned16(t.A) &&
                         (!t.h0 || aligned16(t.h0)) && (!t.h_last || aligned16(t.h_last));
    const int64_t rows = static_cast<int64_t>(t.batch) * t.d_inner;
    const bool tma_ok = lane_ok_common && t.N == 16;
    int variant = a.variant;
    if (variant == AFFINESCAN_VARIANT_AUTO) {
        int sms = 0;
        AS_TRY(sm_count(&sms));
        // one row per FP32 lane of the machine; the structured-A paths need far
        // fewer instructions per row-step, so they pay off from one warp per sub-partition
        const int64_t lane_row_min_rows = static_cast<int64_t>(sms) * 128;
        // very few rows and at least a few tiles per row: parallelise L across CTAs with the
        // decoupled look-back carry.  CHUNKED pays a second exp per state-step, so its time grows
        // with rows * L (~3.3e-8 ms per element) while warp_row_tma's is the serial chain of a
        // row's tiles (~2.7 us each) as long as the rows fit one wave: measured crossover at
        // ~200 rows on 148 SMs (64 rows x 2^20: 2.65 against 7.39 ms; 256 x 2^16: 0.58 against 0.48)
        const bool few_rows = rows * 148 <= static_cast<int64_t>(sms) * 192;
        // general A: lanes = rows (sequential in L) against lanes = timesteps (warp_row_tma, measured
        // ~3.03 cycles per timestep per row and SM, over whole warp tiles of 32 K timesteps):
        // whichever the model says is faster (lane_row only when clearly so: warp_row_tma's cost
        // is not linear in the row count below a few CTAs per SM)
        int g_unused = 0;
        bool lane_wins = rows >= lane_row_min_rows;
        if (a.a_structure == AFFINESCAN_A_GENERAL && lane_ok) {
            const int64_t tile_t = TmaShape<T>::S::kTileT;
            const int64_t padded = (t.L + tile_t - 1) / tile_t * tile_t;
            const double c_tma = 3.03 * static_cast<double>(rows) / sms *
                                     (static_cast<double>(padded) / static_cast<double>(t.L)) + 8.0;
            lane_wins = static_cast<double>(lane_grid_cost(rows, t.d_inner, sms, sizeof(T) == 4,
                                                           &g_unused)) < 0.85 * c_tma;
        }
        if (lane_ok && lane_wins) variant = AFFINESCAN_SELECTIVE_LANE_ROW;
        else if (tma_ok && few_rows && t.L >= kChunkedMinL && !deterministic_auto())
            variant = AFFINESCAN_SELECTIVE_CHUNKED;
        else if (tma_ok && t.L >= kWarpRowTmaMinL) variant = AFFINESCAN_SELECTIVE_WARP_ROW_TMA;
        else variant = AFFINESCAN_SELECTIVE_WARP_ROW;
    }
    int st;
    switch (variant) {
    case AFFINESCAN_SELECTIVE_WARP_ROW:
        st = launch_warp_row<T>(t, vec_ok, stream);
        break;
    case AFFINESCAN_SELECTIVE_WARP_ROW_TMA:
        if (!tma_ok) return AFFINESCAN_ERR_UNSUPPORTED;
        st = launch_warp_row_tma<T>(t, stream);
        break;
    case AFFINESCAN_SELECTIVE_CHUNKED:
        if (!tma_ok) return AFFINESCAN_ERR_UNSUPPORTED;
        st = launch_chunked<T>(t, stream);
        break;
    case AFFINESCAN_SELECTIVE_LANE_ROW:
        if (!lane_ok) return AFFINESCAN_ERR_UNSUPPORTED;
        st = launch_lane_row<T>(t, a.a_structure, stream);
        break;
    default:
        return AFFINESCAN_ERR_UNSUPPORTED;
    }
    if (st == AFFINESCAN_OK) set_last_variant(variant);
    return st;
}

// ---------------------------------------------------------------- L-sharded scan
// P[row][n] = prod_t a_t[row][n] over the slice = 2^(A2[d,n] * sum_t delta[row,t]): one warp per
// row sums delta (coalesced), then lane n raises.  The U half of the slice aggregate is the
// h_last of a scan from h0 = 0 (selective_scan_impl with y == NULL).
template <typename T>
__global__ void __launch_bounds__(256)
slice_decay_kernel(const T* __restrict__ delta, const float* __restrict__ A, float* __restrict__ P,
                   long long rows, int d_inner, int N, long long L)
{
    const int lane = threadIdx.x & 31;
    const long long row = static_cast<long long>(blockIdx.x) * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= rows) return;
    const T* dr = delta + row * L;
    float s = 0.0f;
    for (long long t = lane; t < L; t += 32) {
        float v[1];
        Access<T, 1, true>::load(dr + t, v);
        s += v[0];
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(kFullMask, s, o);
    const int d = static_cast<int>(row % d_inner);
    for (int n = lane; n < N; n += 32)
        P[row * N + n] = ex2_approx(s * (__ldg(A + static_cast<long long>(d) * N + n) * kLog2e));
}

// h_in = state entering the slice of rank `rank`: fold of the aggregates of ranks 0..rank-1 in
// order, (P_j, U_j) (+) ... (+) (P_0, U_0) applied to h0 (Eq.7).
__global__ void compose_carry_kernel(const float* __restrict__ P_all, const float* __restrict__ U_all,
                                     const float* __restrict__ h0, float* __restrict__ h_in,
                                     int rank, long long n)
{
    const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float h = h0 ? h0[i] : 0.0f;
    for (int j = 0; j < rank; ++j) h = fmaf(P_all[j * n + i], h, U_all[j * n + i]);
    h_in[i] = h;
}

}  // namespace

int slice_aggregate_impl(const SelectiveArgs& a, float* P, float* U, void* cuda_stream)
{
    if (a.io_dtype != AFFINESCAN_F32 && a.io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (a.batch < 0 || a.d_inner < 0 || a.L < 0) return AFFINESCAN_ERR_SHAPE;
    if (a.N < 1 || a.N > AFFINESCAN_MAX_N) return AFFINESCAN_ERR_UNSUPPORTED;
    const int64_t rows = static_cast<int64_t>(a.batch) * a.d_inner;
    if (rows == 0) return AFFINESCAN_OK;
    if (!P || !U || !a.A || (a.L > 0 && !a.delta)) return AFFINESCAN_ERR_NULL;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int64_t blocks = (rows + 7) / 8;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    if (a.io_dtype == AFFINESCAN_F32)
        slice_decay_kernel<float><<<static_cast<unsigned>(blocks), 256, 0, stream>>>(
            static_cast<const float*>(a.delta), a.A, P, rows, a.d_inner, a.N, a.L);
    else
        slice_decay_kernel<bf16><<<static_cast<unsigned>(blocks), 256, 0, stream>>>(
            static_cast<const bf16*>(a.delta), a.A, P, rows, a.d_inner, a.N, a.L);
    AS_TRY(after_launch());
    SelectiveArgs s = a;  // U = h_last of the slice scanned from h0 = 0, y not stored
    s.h0 = nullptr;
    s.y = nullptr;
    s.h_last = U;
    return selective_scan_impl(s, cuda_stream);
}

int compose_carry_impl(const float* P_all, const float* U_all, const float* h0, float* h_in,
                       int rank, int world, int64_t n, void* cuda_stream)
{
    if (n < 0 || world < 1 || rank < 0 || rank >= world) return AFFINESCAN_ERR_SHAPE;
    if (n == 0) return AFFINESCAN_OK;
    if (!h_in || (rank > 0 && (!P_all || !U_all))) return AFFINESCAN_ERR_NULL;
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    compose_carry_kernel<<<static_cast<unsigned>(blocks), 256, 0,
                           static_cast<cudaStream_t>(cuda_stream)>>>(P_all, U_all, h0, h_in, rank, n);
    return after_launch();
}

namespace {
}  // namespace

int set_lane_row_option(int key, int value)
{
    switch (key) {
    case AFFINESCAN_OPT_LANE_ROW_G:
        if (value != -1 && (value < 1 || value > 3)) return AFFINESCAN_ERR_UNSUPPORTED;
        g_opt_lane_row_g.store(value);
        return AFFINESCAN_OK;
    case AFFINESCAN_OPT_LANE_ROW_POLY16:
        if (value != -1 && value != 0 && value != 4) return AFFINESCAN_ERR_UNSUPPORTED;
        g_opt_lane_row_poly16.store(value);
        return AFFINESCAN_OK;
    default: return AFFINESCAN_ERR_UNSUPPORTED;
    }
}

int selective_scan_impl(const SelectiveArgs& a, void* cuda_stream)
{
    set_last_variant(0);
    if (a.io_dtype != AFFINESCAN_F32 && a.io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (a.batch < 0 || a.d_inner < 0 || a.L < 0) return AFFINESCAN_ERR_SHAPE;
    if (a.N < 1 || a.N > AFFINESCAN_MAX_N) return AFFINESCAN_ERR_UNSUPPORTED;
    if (a.a_structure < AFFINESCAN_A_GENERAL || a.a_structure > AFFINESCAN_A_POWERS)
        return AFFINESCAN_ERR_UNSUPPORTED;
    int64_t rows = 0, total = 0, bnl = 0;
    if (mul_overflows(a.batch, a.d_inner, &rows) || mul_overflows(rows, a.L, &total) ||
        mul_overflows(static_cast<int64_t>(a.batch) * a.N, a.L, &bnl) ||
        total > (std::numeric_limits<int64_t>::max() >> 3) ||
        bnl > (std::numeric_limits<int64_t>::max() >> 3))
        return AFFINESCAN_ERR_SHAPE;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (rows == 0) return AFFINESCAN_OK;
    if (a.L == 0) return fill_h_last(a.h0, a.h_last, rows * a.N, stream);
    // y == NULL is allowed when h_last is wanted: the aggregate-only call of the L-sharded scan
    if (!a.x || !a.delta || !a.A || !a.B || !a.C || (!a.y && !a.h_last)) return AFFINESCAN_ERR_NULL;
    return a.io_dtype == AFFINESCAN_F32 ? selective_dispatch<float>(a, stream)
                                        : selective_dispatch<bf16>(a, stream);
}

}  // namespace affinescan_host
