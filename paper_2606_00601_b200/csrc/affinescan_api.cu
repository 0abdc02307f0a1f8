// affinescan_api.cu — C-ABI boundary and host launch layer of libaffinescan
// (include/affinescan.h).  Validates arguments, picks a kernel variant from the shape,
// and enqueues the kernels on the caller's stream.  No torch types, no exceptions.
#include "../../include/affinescan.h"

#include <atomic>
#include <cstdint>
#include <limits>
#include <map>
#include <mutex>
#include <utility>
#include <vector>

#include "affine_scan.cuh"
#include "selective_scan_lane_row.cuh"
#include "selective_scan_warp_row.cuh"
#include "selective_scan_warp_row_tma.cuh"

namespace {

using namespace affinescan;
using bf16 = __nv_bfloat16;

thread_local int tl_last_cuda_error = 0;
thread_local int tl_last_variant = 0;
std::atomic<int64_t> g_launches{0};

int cuda_fail(cudaError_t e)
{
    tl_last_cuda_error = static_cast<int>(e);
    (void)cudaGetLastError();  // clear the sticky-less error state
    return AFFINESCAN_ERR_CUDA;
}
#define AS_CUDA(call)                                     \
    do {                                                  \
        const cudaError_t e__ = (call);                   \
        if (e__ != cudaSuccess) return cuda_fail(e__);    \
    } while (0)

int after_launch()
{
    g_launches.fetch_add(1, std::memory_order_relaxed);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? AFFINESCAN_OK : cuda_fail(e);
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

bool mul_overflows(int64_t a, int64_t b, int64_t* out)
{
    return __builtin_mul_overflow(a, b, out);
}

// ---------------------------------------------------------------- device buffer caches
struct Buffer {
    void* ptr = nullptr;
    size_t bytes = 0;
};
std::mutex g_mu;
std::mutex g_host_mu;  // the _host entry points share the per-device staging buffers
std::map<std::pair<int, void*>, Buffer> g_scratch;  // (device, stream) -> look-back scratch
std::map<std::pair<int, int>, Buffer> g_staging;    // (device, slot)   -> host-API staging

int grow(Buffer& b, size_t bytes)
{
    if (b.bytes >= bytes) return AFFINESCAN_OK;
    if (b.ptr) {
        AS_CUDA(cudaDeviceSynchronize());  // an earlier call on this stream may still use it
        AS_CUDA(cudaFree(b.ptr));
        b.ptr = nullptr;
        b.bytes = 0;
    }
    const size_t want = bytes + bytes / 4 + 256;
    AS_CUDA(cudaMalloc(&b.ptr, want));
    b.bytes = want;
    return AFFINESCAN_OK;
}

int get_scratch(cudaStream_t stream, size_t bytes, void** out)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_mu);
    Buffer& b = g_scratch[{dev, static_cast<void*>(stream)}];
    const int st = grow(b, bytes);
    if (st != AFFINESCAN_OK) return st;
    *out = b.ptr;
    return AFFINESCAN_OK;
}

int get_staging(int slot, size_t bytes, void** out)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_mu);
    Buffer& b = g_staging[{dev, slot}];
    const int st = grow(b, bytes ? bytes : 1);
    if (st != AFFINESCAN_OK) return st;
    *out = b.ptr;
    return AFFINESCAN_OK;
}

size_t elt_size(int io_dtype) { return io_dtype == AFFINESCAN_BF16 ? 2 : 4; }

// ============================================================== affine_scan dispatch
constexpr int kAffJ = 4;       // 128-bit vectors per thread per tile
constexpr int kAffWarps = 8;   // 256 threads
constexpr int kAffLookbackWarps = 8;   // (16 warps = 8192-element tiles measured the same on long L,
                                       // slower on short L)
constexpr int kAffLookbackJ = 4;  // look-back tiles of 4096 elements (J = 8: 202 registers, 2.5 TB/s)
constexpr int64_t kAffWarpSeqMinSeq = 148 * 64;  // >= 64 independent warps per SM
constexpr int64_t kAffCtaLoopMinSeq = 148 * 4;   // >= 4 CTAs of 8 warps per SM
constexpr int64_t kAffCtaLoopMinL = 8192;        // at least two CTA tiles per sequence

template <typename T, int VEC>
int launch_affine_lookback(const T* a, const T* u, const float* h0, T* h, float* h_last,
                           int64_t num_seq, int64_t L, cudaStream_t stream)
{
    // 4096-element tiles for both io dtypes (64 B of a and of u per thread fit 64 registers)
    constexpr int kJ = VEC == 8 ? kAffLookbackJ / 2 : kAffLookbackJ;
    constexpr int kTile = kAffLookbackWarps * 32 * VEC * kJ;
    const int64_t total = num_seq * L;
    const int64_t ntiles = (total + kTile - 1) / kTile;
    if (ntiles > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    void* scratch = nullptr;
    const size_t desc_bytes = static_cast<size_t>(ntiles) * 16;
    const int st = get_scratch(stream, desc_bytes + 16, &scratch);
    if (st != AFFINESCAN_OK) return st;
    AS_CUDA(cudaMemsetAsync(scratch, 0, desc_bytes + 16, stream));
    auto* desc = static_cast<unsigned long long*>(scratch);
    auto* ticket = reinterpret_cast<unsigned*>(static_cast<unsigned char*>(scratch) + desc_bytes);
    affine_scan_lookback_kernel<T, VEC, kJ, kAffLookbackWarps>
        <<<static_cast<unsigned>(ntiles), kAffLookbackWarps * 32, 0, stream>>>(a, u, h0, h, h_last, total, L,
                                                                      desc, ticket);
    return after_launch();
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
    // decoupled look-back carry.
    if (variant == AFFINESCAN_VARIANT_AUTO) {
        if (num_seq >= kAffCtaLoopMinSeq && L >= kAffCtaLoopMinL)
            variant = AFFINESCAN_AFFINE_CTA_LOOP;
        else if (num_seq >= kAffWarpSeqMinSeq) variant = AFFINESCAN_AFFINE_WARP_SEQ;
        else if (L <= kAffCtaLoopMinL) variant = AFFINESCAN_AFFINE_CTA_LOOP;  // latency-bound:
        else variant = AFFINESCAN_AFFINE_LOOKBACK;  // no memset, no ticket (cfg1 9.7 -> 6.6 us)
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
    if (st == AFFINESCAN_OK) tl_last_variant = variant;
    return st;
}

__global__ void fill_h_last_kernel(const float* __restrict__ h0, float* __restrict__ h_last,
                                   long long n)
{
    const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < n) h_last[i] = h0 ? h0[i] : 0.0f;
}

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
    tl_last_variant = 0;
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

// ============================================================== selective_scan dispatch
constexpr int kSmCount = 148;
constexpr int kWarpRowTmaRowsPerWarpF32 = 1;
constexpr int kWarpRowTmaMaxWarps2 = 7;    // two rows per warp: (7+1) warps x 32 x <= 255 registers
constexpr int kWarpRowTmaMaxWarps = 11;   // warp_row_tma: rows per CTA (+1 producer warp = 384 threads)
constexpr int64_t kWarpRowTmaMinL = 1024; // below two warp tiles the plain warp_row is as good
constexpr int kSelWarps = 4;        // warp_row: rows per CTA
constexpr int kLaneRowTc = 32;      // lane_row: timesteps per staged B/C tile
constexpr int kLaneRowWarps = 4;    // lane_row: warps per CTA (autonomous)
constexpr int kLaneRowPairsPerPass = 2;   // packed pairs per pass (ILP of the MUFU burst)
constexpr bool kLaneRowPipelined = false;  // ablation: 2^x of pass q+1 between the chain steps of pass q (0.407 vs 0.348 ms)
constexpr int kLaneRowDefaultG = 1;       // lanes per row (r01b sweep: profiles/)
constexpr int kLaneRowDefaultPoly16 = 4;  // sixteenths of the exps done on the fma pipe
constexpr int64_t kLaneRowMinRows = 148 * 32 * 4;  // one row per FP32 lane of the machine

template <typename T, int VEC, int NV>
int launch_warp_row(const T* x, const T* delta, const float* A, const T* B, const T* C,
                    const float* D, const float* h0, T* y, float* h_last, int batch, int d_inner,
                    int N, int64_t L, cudaStream_t stream)
{
    const int64_t rows = static_cast<int64_t>(batch) * d_inner;
    const int64_t blocks = (rows + kSelWarps - 1) / kSelWarps;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    selective_scan_warp_row_kernel<T, VEC, NV, kSelWarps>
        <<<static_cast<unsigned>(blocks), kSelWarps * 32, 0, stream>>>(x, delta, A, B, C, D, h0, y,
                                                                       h_last, batch, d_inner, N, L);
    return after_launch();
}

// Tuning knobs of the lane_row schedule (affinescan_set_option); -1 = choose from the shape.
std::atomic<int> g_opt_lane_row_g{-1};
std::atomic<int> g_opt_lane_row_poly16{-1};

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

// Tensor map over a [batch*N, L] io-dtype matrix (B or C), box = {box_t timesteps, N rows}.
template <typename T>
int make_bc_tensor_map(CUtensorMap* map, const T* base, int64_t rows, int64_t L, int box_t, int N)
{
    EncodeTiledFn encode = nullptr;
    const int st = get_encode_tiled(&encode);
    if (st != AFFINESCAN_OK) return st;
    const cuuint64_t dims[2] = {static_cast<cuuint64_t>(L), static_cast<cuuint64_t>(rows)};
    const cuuint64_t strides[1] = {static_cast<cuuint64_t>(L) * sizeof(T)};
    const cuuint32_t box[2] = {static_cast<cuuint32_t>(box_t), static_cast<cuuint32_t>(N)};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode(map, sizeof(T) == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                                  : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                              2, const_cast<T*>(base), dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? AFFINESCAN_OK : cuda_fail(cudaErrorInvalidValue);
}

template <typename T, int G, int F16>
int launch_lane_row_inst(const T* x, const T* delta, const float* A, const T* B, const T* C,
                         const float* D, const float* h0, T* y, float* h_last, int batch,
                         int d_inner, int64_t L, cudaStream_t stream)
{
    // polynomial degree per io dtype: DESIGN.md §7 (tolerance argument)
    constexpr int kDeg = sizeof(T) == 2 ? 3 : 5;
    using S = LaneRowSmem<T, kLaneRowTc>;
    constexpr int kNp = 8 / G;
    constexpr int kPp = kLaneRowPairsPerPass < kNp ? kLaneRowPairsPerPass : kNp;
    auto kern = selective_scan_lane_row_kernel<T, G, kLaneRowTc, kLaneRowWarps, F16, kDeg, kPp,
                                               kLaneRowPipelined>;
    constexpr int smem = S::kPerWarp * kLaneRowWarps;
    static std::atomic<unsigned> configured{0};  // bit per device
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    if (!(configured.load() & (1u << (dev & 31)))) {
        AS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        configured.fetch_or(1u << (dev & 31));
    }
    CUtensorMap mapB, mapC;
    int st = make_bc_tensor_map<T>(&mapB, B, static_cast<int64_t>(batch) * 16, L, kLaneRowTc, 16);
    if (st != AFFINESCAN_OK) return st;
    st = make_bc_tensor_map<T>(&mapC, C, static_cast<int64_t>(batch) * 16, L, kLaneRowTc, 16);
    if (st != AFFINESCAN_OK) return st;
    const int64_t rows = static_cast<int64_t>(batch) * d_inner;
    const int64_t warps = rows / (32 / G);
    const int64_t blocks = (warps + kLaneRowWarps - 1) / kLaneRowWarps;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    kern<<<static_cast<unsigned>(blocks), kLaneRowWarps * 32, smem, stream>>>(
        x, delta, A, mapB, mapC, D, h0, y, h_last, batch, d_inner, L);
    return after_launch();
}

template <typename T, int G>
int launch_lane_row_g(int poly16, const T* x, const T* delta, const float* A, const T* B,
                      const T* C, const float* D, const float* h0, T* y, float* h_last, int batch,
                      int d_inner, int64_t L, cudaStream_t stream)
{
#define AS_LANE_ROW_CASE(F)                                                                      \
    case F:                                                                                      \
        return launch_lane_row_inst<T, G, F>(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, \
                                             L, stream)
    switch (poly16) {
        AS_LANE_ROW_CASE(0);
        AS_LANE_ROW_CASE(3);
        AS_LANE_ROW_CASE(4);
        AS_LANE_ROW_CASE(5);
        AS_LANE_ROW_CASE(6);
    default: return AFFINESCAN_ERR_UNSUPPORTED;
    }
#undef AS_LANE_ROW_CASE
}

template <typename T>
int launch_lane_row(const T* x, const T* delta, const float* A, const T* B, const T* C,
                    const float* D, const float* h0, T* y, float* h_last, int batch, int d_inner,
                    int64_t L, cudaStream_t stream)
{
    int G = g_opt_lane_row_g.load(std::memory_order_relaxed);
    int poly16 = g_opt_lane_row_poly16.load(std::memory_order_relaxed);
    if (G < 0) G = kLaneRowDefaultG;
    if (poly16 < 0) poly16 = kLaneRowDefaultPoly16;
    switch (G) {
    case 1:
        return launch_lane_row_g<T, 1>(poly16, x, delta, A, B, C, D, h0, y, h_last, batch, d_inner,
                                       L, stream);
    case 2:
        return launch_lane_row_g<T, 2>(poly16, x, delta, A, B, C, D, h0, y, h_last, batch, d_inner,
                                       L, stream);
    case 4:
        return launch_lane_row_g<T, 4>(poly16, x, delta, A, B, C, D, h0, y, h_last, batch, d_inner,
                                       L, stream);
    default: return AFFINESCAN_ERR_UNSUPPORTED;
    }
}

template <typename T>
int launch_warp_row_tma(const T* x, const T* delta, const float* A, const T* B, const T* C,
                        const float* D, const float* h0, T* y, float* h_last, int batch,
                        int d_inner, int64_t L, cudaStream_t stream)
{
    constexpr int kVec = Io<T>::kVec;
    // odd: conflict-free LDS.128 (K = 12 fp32 / 24 bf16 timesteps per lane; K = 20 with one
    // chain measured slower: cfg4 0.906 vs 0.818 ms)
    constexpr int kNv = 3;
    using S = WarpRowTmaSmem<T, kNv * kVec>;
    // chains per warp = NU states x RW rows.  fp32 io: two states of one row (two rows per warp
    // sharing every LDS.128 of B_t/C_t halve the shared-memory traffic but leave 6 warps per SM:
    // cfg4 1.14 vs 0.82 ms); bf16 io: K = 24 leaves registers for one chain only.
    constexpr int kRw = sizeof(T) == 2 ? 1 : kWarpRowTmaRowsPerWarpF32;
    constexpr int kNu = (sizeof(T) == 2 || kRw == 2) ? 1 : 2;
    auto kern = selective_scan_warp_row_tma_kernel<T, kVec, kNv, kNu, kRw>;
    static std::atomic<unsigned> configured{0};  // bit per device
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    if (!(configured.load() & (1u << (dev & 31)))) {
        AS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::kBytes));
        configured.fetch_or(1u << (dev & 31));
    }
    CUtensorMap mapB, mapC;
    int st = make_bc_tensor_map<T>(&mapB, B, static_cast<int64_t>(batch) * 16, L, S::kBoxT, 16);
    if (st != AFFINESCAN_OK) return st;
    st = make_bc_tensor_map<T>(&mapC, C, static_cast<int64_t>(batch) * 16, L, S::kBoxT, 16);
    if (st != AFFINESCAN_OK) return st;
    // R rows (warps) of one batch per CTA, sized so that one wave of CTAs covers all rows when
    // they fit (cfg2/cfg4: 1536 rows -> 140 CTAs of 11 warps on 148 SMs)
    const int slots = kSmCount / batch > 0 ? kSmCount / batch : 1;
    const int max_warps = kRw == 1 ? kWarpRowTmaMaxWarps : kWarpRowTmaMaxWarps2;
    int R = ((d_inner + slots - 1) / slots + kRw - 1) / kRw;  // consumer warps per CTA
    R = R < 1 ? 1 : (R > max_warps ? max_warps : R);
    const int ctas_per_batch = (d_inner + R * kRw - 1) / (R * kRw);
    const int64_t blocks = static_cast<int64_t>(batch) * ctas_per_batch;
    if (blocks > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    kern<<<static_cast<unsigned>(blocks), (R + 1) * 32, S::kBytes, stream>>>(
        x, delta, A, mapB, mapC, D, h0, y, h_last, batch, d_inner, ctas_per_batch, L);
    return after_launch();
}

template <typename T>
int selective_dispatch(const void* x_, const void* delta_, const float* A, const void* B_,
                       const void* C_, const float* D, const float* h0, void* y_, float* h_last,
                       int batch, int d_inner, int N, int64_t L, int variant, cudaStream_t stream)
{
    const T* x = static_cast<const T*>(x_);
    const T* delta = static_cast<const T*>(delta_);
    const T* B = static_cast<const T*>(B_);
    const T* C = static_cast<const T*>(C_);
    T* y = static_cast<T*>(y_);
    constexpr int kVec = Io<T>::kVec;
    const bool vec_ok = (L % kVec == 0) && aligned16(x) && aligned16(delta) && aligned16(B) &&
                        aligned16(C) && aligned16(y);
    const bool lane_ok_common = vec_ok && L < (1LL << 31) - 4096;  // TMA coordinates are int32
    const bool lane_ok = lane_ok_common && N == 16 && (d_inner % 32 == 0) && aligned16(A) &&
                         (!h0 || aligned16(h0)) && (!h_last || aligned16(h_last));
    const int64_t rows = static_cast<int64_t>(batch) * d_inner;
    const bool tma_ok = lane_ok_common && N == 16;
    if (variant == AFFINESCAN_VARIANT_AUTO) {
        if (lane_ok && rows >= kLaneRowMinRows) variant = AFFINESCAN_SELECTIVE_LANE_ROW;
        else if (tma_ok && L >= kWarpRowTmaMinL) variant = AFFINESCAN_SELECTIVE_WARP_ROW_TMA;
        else variant = AFFINESCAN_SELECTIVE_WARP_ROW;
    }
    int st;
    switch (variant) {
    case AFFINESCAN_SELECTIVE_WARP_ROW:
        if (vec_ok)
            st = launch_warp_row<T, kVec, 16 / kVec>(x, delta, A, B, C, D, h0, y, h_last, batch,
                                                     d_inner, N, L, stream);
        else
            st = launch_warp_row<T, 1, 4>(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N, L,
                                          stream);
        break;
    case AFFINESCAN_SELECTIVE_WARP_ROW_TMA:
        if (!tma_ok) return AFFINESCAN_ERR_UNSUPPORTED;
        st = launch_warp_row_tma<T>(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, L, stream);
        break;
    case AFFINESCAN_SELECTIVE_LANE_ROW:
        if (!lane_ok) return AFFINESCAN_ERR_UNSUPPORTED;
        st = launch_lane_row<T>(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, L, stream);
        break;
    default:
        return AFFINESCAN_ERR_UNSUPPORTED;
    }
    if (st == AFFINESCAN_OK) tl_last_variant = variant;
    return st;
}

int selective_scan_impl(const void* x, const void* delta, const float* A, const void* B,
                        const void* C, const float* D, const float* h0, void* y, float* h_last,
                        int batch, int d_inner, int N, int64_t L, int io_dtype, int variant,
                        void* cuda_stream)
{
    tl_last_variant = 0;
    if (io_dtype != AFFINESCAN_F32 && io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (batch < 0 || d_inner < 0 || L < 0) return AFFINESCAN_ERR_SHAPE;
    if (N < 1 || N > AFFINESCAN_MAX_N) return AFFINESCAN_ERR_UNSUPPORTED;
    int64_t rows = 0, total = 0, bnl = 0;
    if (mul_overflows(batch, d_inner, &rows) || mul_overflows(rows, L, &total) ||
        mul_overflows(static_cast<int64_t>(batch) * N, L, &bnl) ||
        total > (std::numeric_limits<int64_t>::max() >> 3) ||
        bnl > (std::numeric_limits<int64_t>::max() >> 3))
        return AFFINESCAN_ERR_SHAPE;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (rows == 0) return AFFINESCAN_OK;
    if (L == 0) return fill_h_last(h0, h_last, rows * N, stream);
    if (!x || !delta || !A || !B || !C || !y) return AFFINESCAN_ERR_NULL;
    return io_dtype == AFFINESCAN_F32
               ? selective_dispatch<float>(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N,
                                           L, variant, stream)
               : selective_dispatch<bf16>(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N,
                                          L, variant, stream);
}

// ---------------------------------------------------------------- host-buffer helpers
struct Staged {
    void* dev = nullptr;
};

int stage_in(int slot, const void* host, size_t bytes, cudaStream_t stream, void** dev)
{
    *dev = nullptr;
    if (!host) return AFFINESCAN_OK;
    const int st = get_staging(slot, bytes, dev);
    if (st != AFFINESCAN_OK) return st;
    if (bytes) AS_CUDA(cudaMemcpyAsync(*dev, host, bytes, cudaMemcpyHostToDevice, stream));
    return AFFINESCAN_OK;
}

// Copy-in / copy-out streams and events of the pipelined _host entry point (per device).
struct HostPipe {
    cudaStream_t in = nullptr, out = nullptr;
    cudaEvent_t start = nullptr;
    std::vector<cudaEvent_t> in_done, k_done;
};
std::map<int, HostPipe> g_pipes;

int get_host_pipe(HostPipe** out)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_mu);
    HostPipe& p = g_pipes[dev];
    if (!p.in) {
        AS_CUDA(cudaStreamCreateWithFlags(&p.in, cudaStreamNonBlocking));
        AS_CUDA(cudaStreamCreateWithFlags(&p.out, cudaStreamNonBlocking));
        AS_CUDA(cudaEventCreateWithFlags(&p.start, cudaEventDisableTiming));
    }
    *out = &p;
    return AFFINESCAN_OK;
}

int stage_out_alloc(int slot, const void* host, size_t bytes, void** dev)
{
    *dev = nullptr;
    if (!host) return AFFINESCAN_OK;
    return get_staging(slot, bytes, dev);
}

}  // namespace

// =================================================================== exported C ABI
extern "C" {

int affine_scan(const void* a, const void* u, const float* h0, void* h, float* h_last,
                int64_t num_seq, int64_t L, int io_dtype, void* cuda_stream)
{
    return affine_scan_impl(a, u, h0, h, h_last, num_seq, L, io_dtype, AFFINESCAN_VARIANT_AUTO,
                            cuda_stream);
}

int affine_scan_ex(const void* a, const void* u, const float* h0, void* h, float* h_last,
                   int64_t num_seq, int64_t L, int io_dtype, int variant, void* cuda_stream)
{
    return affine_scan_impl(a, u, h0, h, h_last, num_seq, L, io_dtype, variant, cuda_stream);
}

int affine_scan_host(const void* a, const void* u, const float* h0, void* h, float* h_last,
                     int64_t num_seq, int64_t L, int io_dtype, void* cuda_stream)
{
    if (io_dtype != AFFINESCAN_F32 && io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (num_seq < 0 || L < 0) return AFFINESCAN_ERR_SHAPE;
    int64_t total = 0;
    if (mul_overflows(num_seq, L, &total) || total > (std::numeric_limits<int64_t>::max() >> 3))
        return AFFINESCAN_ERR_SHAPE;
    if (total > 0 && (!a || !u || !h)) return AFFINESCAN_ERR_NULL;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    std::lock_guard<std::mutex> host_lock(g_host_mu);
    const size_t eb = static_cast<size_t>(total) * elt_size(io_dtype);
    const size_t sb = static_cast<size_t>(num_seq) * sizeof(float);
    void *da, *du, *dh0, *dh, *dhl;
    int st;
    // same three-stage pipeline as selective_scan_fwd_host, over chunks of whole sequences
    if ((st = get_staging(0, eb, &da)) != AFFINESCAN_OK) return st;
    if ((st = get_staging(1, eb, &du)) != AFFINESCAN_OK) return st;
    if ((st = stage_in(2, h0, sb, stream, &dh0)) != AFFINESCAN_OK) return st;
    if ((st = stage_out_alloc(3, h, eb, &dh)) != AFFINESCAN_OK) return st;
    if ((st = stage_out_alloc(4, h_last, sb, &dhl)) != AFFINESCAN_OK) return st;
    if (total == 0) {  // nothing to scan: h_last <- h0 (or 0)
        st = affine_scan_impl(da, du, static_cast<const float*>(dh0), dh, static_cast<float*>(dhl),
                              num_seq, L, io_dtype, AFFINESCAN_VARIANT_AUTO, cuda_stream);
        if (st != AFFINESCAN_OK) return st;
        if (h_last && sb) AS_CUDA(cudaMemcpyAsync(h_last, dhl, sb, cudaMemcpyDeviceToHost, stream));
        AS_CUDA(cudaStreamSynchronize(stream));
        return AFFINESCAN_OK;
    }
    HostPipe* pipe = nullptr;
    if ((st = get_host_pipe(&pipe)) != AFFINESCAN_OK) return st;
    const size_t seq_bytes = static_cast<size_t>(L) * elt_size(io_dtype);
    int64_t per = static_cast<int64_t>((16u << 20) / seq_bytes) + 1;  // sequences per chunk
    if (per > num_seq) per = num_seq;
    int64_t nchunks = (num_seq + per - 1) / per;
    if (nchunks > 64) {  // bound the number of events
        nchunks = 64;
        per = (num_seq + nchunks - 1) / nchunks;
        nchunks = (num_seq + per - 1) / per;
    }
    if (static_cast<int64_t>(pipe->in_done.size()) < nchunks) {
        const size_t old = pipe->in_done.size();
        pipe->in_done.resize(nchunks);
        pipe->k_done.resize(nchunks);
        for (size_t i = old; i < pipe->in_done.size(); ++i) {
            AS_CUDA(cudaEventCreateWithFlags(&pipe->in_done[i], cudaEventDisableTiming));
            AS_CUDA(cudaEventCreateWithFlags(&pipe->k_done[i], cudaEventDisableTiming));
        }
    }
    AS_CUDA(cudaEventRecord(pipe->start, stream));
    AS_CUDA(cudaStreamWaitEvent(pipe->in, pipe->start, 0));
    AS_CUDA(cudaStreamWaitEvent(pipe->out, pipe->start, 0));
    auto at = [](const void* p, size_t bytes) {
        return const_cast<void*>(static_cast<const void*>(static_cast<const unsigned char*>(p) + bytes));
    };
    for (int64_t c = 0; c < nchunks; ++c) {
        const int64_t s0 = c * per;
        const int64_t ns = (s0 + per <= num_seq) ? per : num_seq - s0;
        const size_t eo = seq_bytes * s0, so = sizeof(float) * s0;
        AS_CUDA(cudaMemcpyAsync(at(da, eo), at(a, eo), seq_bytes * ns, cudaMemcpyHostToDevice, pipe->in));
        AS_CUDA(cudaMemcpyAsync(at(du, eo), at(u, eo), seq_bytes * ns, cudaMemcpyHostToDevice, pipe->in));
        AS_CUDA(cudaEventRecord(pipe->in_done[c], pipe->in));
        AS_CUDA(cudaStreamWaitEvent(stream, pipe->in_done[c], 0));
        st = affine_scan_impl(at(da, eo), at(du, eo),
                              dh0 ? static_cast<const float*>(at(dh0, so)) : nullptr, at(dh, eo),
                              dhl ? static_cast<float*>(at(dhl, so)) : nullptr, ns, L, io_dtype,
                              AFFINESCAN_VARIANT_AUTO, cuda_stream);
        if (st != AFFINESCAN_OK) return st;
        AS_CUDA(cudaEventRecord(pipe->k_done[c], stream));
        AS_CUDA(cudaStreamWaitEvent(pipe->out, pipe->k_done[c], 0));
        AS_CUDA(cudaMemcpyAsync(at(h, eo), at(dh, eo), seq_bytes * ns, cudaMemcpyDeviceToHost, pipe->out));
        if (h_last)
            AS_CUDA(cudaMemcpyAsync(at(h_last, so), at(dhl, so), sizeof(float) * ns,
                                    cudaMemcpyDeviceToHost, pipe->out));
    }
    AS_CUDA(cudaStreamSynchronize(pipe->out));
    AS_CUDA(cudaStreamSynchronize(stream));
    return AFFINESCAN_OK;
}

int selective_scan_fwd(const void* x, const void* delta, const float* A, const void* B,
                       const void* C, const float* D, const float* h0, void* y, float* h_last,
                       int batch, int d_inner, int N, int64_t L, int io_dtype, void* cuda_stream)
{
    return selective_scan_impl(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N, L, io_dtype,
                               AFFINESCAN_VARIANT_AUTO, cuda_stream);
}

int selective_scan_fwd_ex(const void* x, const void* delta, const float* A, const void* B,
                          const void* C, const float* D, const float* h0, void* y, float* h_last,
                          int batch, int d_inner, int N, int64_t L, int io_dtype, int variant,
                          void* cuda_stream)
{
    return selective_scan_impl(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N, L, io_dtype,
                               variant, cuda_stream);
}

int selective_scan_fwd_host(const void* x, const void* delta, const float* A, const void* B,
                            const void* C, const float* D, const float* h0, void* y, float* h_last,
                            int batch, int d_inner, int N, int64_t L, int io_dtype,
                            void* cuda_stream)
{
    if (io_dtype != AFFINESCAN_F32 && io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (batch < 0 || d_inner < 0 || L < 0) return AFFINESCAN_ERR_SHAPE;
    if (N < 1 || N > AFFINESCAN_MAX_N) return AFFINESCAN_ERR_UNSUPPORTED;
    int64_t rows = 0, total = 0, bnl = 0;
    if (mul_overflows(batch, d_inner, &rows) || mul_overflows(rows, L, &total) ||
        mul_overflows(static_cast<int64_t>(batch) * N, L, &bnl) ||
        total > (std::numeric_limits<int64_t>::max() >> 3) ||
        bnl > (std::numeric_limits<int64_t>::max() >> 3))
        return AFFINESCAN_ERR_SHAPE;
    if (total > 0 && (!x || !delta || !A || !B || !C || !y)) return AFFINESCAN_ERR_NULL;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    std::lock_guard<std::mutex> host_lock(g_host_mu);
    const size_t es = elt_size(io_dtype);
    const size_t xb = static_cast<size_t>(total) * es;
    const size_t bb = static_cast<size_t>(bnl) * es;
    const size_t ab = static_cast<size_t>(d_inner) * N * sizeof(float);
    const size_t db = static_cast<size_t>(d_inner) * sizeof(float);
    const size_t hb = static_cast<size_t>(rows) * N * sizeof(float);
    void *dx, *dd, *dA, *dB, *dC, *dD, *dh0, *dy, *dhl;
    int st;
    // Device staging (cached, full size), then a three-stage pipeline over batches:
    // H2D of batch b+1 (copy-in stream) || kernel of batch b (caller's stream) || D2H of batch
    // b-1 (copy-out stream).  PCIe is full duplex, so the step costs ~max(H2D, D2H), not the sum.
    if ((st = get_staging(10, xb, &dx)) != AFFINESCAN_OK) return st;
    if ((st = get_staging(11, xb, &dd)) != AFFINESCAN_OK) return st;
    if ((st = stage_in(12, A, ab, stream, &dA)) != AFFINESCAN_OK) return st;
    if ((st = get_staging(13, bb, &dB)) != AFFINESCAN_OK) return st;
    if ((st = get_staging(14, bb, &dC)) != AFFINESCAN_OK) return st;
    if ((st = stage_in(15, D, db, stream, &dD)) != AFFINESCAN_OK) return st;
    if ((st = stage_in(16, h0, hb, stream, &dh0)) != AFFINESCAN_OK) return st;
    if ((st = stage_out_alloc(17, y, xb, &dy)) != AFFINESCAN_OK) return st;
    if ((st = stage_out_alloc(18, h_last, hb, &dhl)) != AFFINESCAN_OK) return st;
    if (total == 0) {
        AS_CUDA(cudaStreamSynchronize(stream));
        return AFFINESCAN_OK;
    }
    HostPipe* pipe = nullptr;
    if ((st = get_host_pipe(&pipe)) != AFFINESCAN_OK) return st;
    // batches per chunk: at least ~16 MB of x per chunk so that copies stay at full PCIe rate
    const size_t xb1 = xb / batch, bb1 = bb / batch, hb1 = hb / batch;
    int per = static_cast<int>((16u << 20) / (xb1 ? xb1 : 1)) + 1;
    if (per > batch) per = batch;
    const int nchunks = (batch + per - 1) / per;
    if (static_cast<int>(pipe->in_done.size()) < nchunks) {
        const size_t old = pipe->in_done.size();
        pipe->in_done.resize(nchunks);
        pipe->k_done.resize(nchunks);
        for (size_t i = old; i < pipe->in_done.size(); ++i) {
            AS_CUDA(cudaEventCreateWithFlags(&pipe->in_done[i], cudaEventDisableTiming));
            AS_CUDA(cudaEventCreateWithFlags(&pipe->k_done[i], cudaEventDisableTiming));
        }
    }
    // the small per-call tensors (A, D, h0) went in on the caller's stream: the copy streams must
    // not overtake an earlier call's use of the staging buffers either
    AS_CUDA(cudaEventRecord(pipe->start, stream));
    AS_CUDA(cudaStreamWaitEvent(pipe->in, pipe->start, 0));
    AS_CUDA(cudaStreamWaitEvent(pipe->out, pipe->start, 0));
    auto off = [](const void* p, size_t bytes) {
        return static_cast<const void*>(static_cast<const unsigned char*>(p) + bytes);
    };
    auto offm = [](void* p, size_t bytes) {
        return static_cast<void*>(static_cast<unsigned char*>(p) + bytes);
    };
    for (int c = 0; c < nchunks; ++c) {
        const int b0 = c * per;
        const int nb = (b0 + per <= batch) ? per : batch - b0;
        const size_t xo = xb1 * b0, bo = bb1 * b0, ho = hb1 * b0;
        AS_CUDA(cudaMemcpyAsync(offm(dx, xo), off(x, xo), xb1 * nb, cudaMemcpyHostToDevice, pipe->in));
        AS_CUDA(cudaMemcpyAsync(offm(dd, xo), off(delta, xo), xb1 * nb, cudaMemcpyHostToDevice, pipe->in));
        AS_CUDA(cudaMemcpyAsync(offm(dB, bo), off(B, bo), bb1 * nb, cudaMemcpyHostToDevice, pipe->in));
        AS_CUDA(cudaMemcpyAsync(offm(dC, bo), off(C, bo), bb1 * nb, cudaMemcpyHostToDevice, pipe->in));
        AS_CUDA(cudaEventRecord(pipe->in_done[c], pipe->in));
        AS_CUDA(cudaStreamWaitEvent(stream, pipe->in_done[c], 0));
        st = selective_scan_impl(offm(dx, xo), offm(dd, xo), static_cast<const float*>(dA),
                                 offm(dB, bo), offm(dC, bo), static_cast<const float*>(dD),
                                 dh0 ? static_cast<const float*>(offm(dh0, ho)) : nullptr,
                                 offm(dy, xo), dhl ? static_cast<float*>(offm(dhl, ho)) : nullptr, nb,
                                 d_inner, N, L, io_dtype, AFFINESCAN_VARIANT_AUTO, cuda_stream);
        if (st != AFFINESCAN_OK) return st;
        AS_CUDA(cudaEventRecord(pipe->k_done[c], stream));
        AS_CUDA(cudaStreamWaitEvent(pipe->out, pipe->k_done[c], 0));
        AS_CUDA(cudaMemcpyAsync(offm(y, xo), off(dy, xo), xb1 * nb, cudaMemcpyDeviceToHost, pipe->out));
        if (h_last)
            AS_CUDA(cudaMemcpyAsync(offm(h_last, ho), off(dhl, ho), hb1 * nb, cudaMemcpyDeviceToHost,
                                    pipe->out));
    }
    AS_CUDA(cudaStreamSynchronize(pipe->out));
    AS_CUDA(cudaStreamSynchronize(stream));
    return AFFINESCAN_OK;
}

const char* affinescan_status_string(int status)
{
    switch (status) {
    case AFFINESCAN_OK: return "ok";
    case AFFINESCAN_ERR_NULL: return "a required pointer is NULL";
    case AFFINESCAN_ERR_SHAPE: return "negative or overflowing shape";
    case AFFINESCAN_ERR_DTYPE: return "unknown io dtype";
    case AFFINESCAN_ERR_UNSUPPORTED: return "unsupported N, variant or shape for the forced variant";
    case AFFINESCAN_ERR_CUDA: return "CUDA runtime error (see affinescan_last_cuda_error)";
    default: return "unknown status";
    }
}

int affinescan_last_cuda_error(void) { return tl_last_cuda_error; }
int affinescan_last_variant(void) { return tl_last_variant; }
int64_t affinescan_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
int affinescan_version(void) { return 100; }

int affinescan_set_option(int key, int value)
{
    switch (key) {
    case AFFINESCAN_OPT_LANE_ROW_G:
        if (value != -1 && value != 1 && value != 2 && value != 4) return AFFINESCAN_ERR_UNSUPPORTED;
        g_opt_lane_row_g.store(value);
        return AFFINESCAN_OK;
    case AFFINESCAN_OPT_LANE_ROW_POLY16:
        if (value != -1 && value != 0 && (value < 3 || value > 6)) return AFFINESCAN_ERR_UNSUPPORTED;
        g_opt_lane_row_poly16.store(value);
        return AFFINESCAN_OK;
    default: return AFFINESCAN_ERR_UNSUPPORTED;
    }
}

int affinescan_release_cache(void)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    AS_CUDA(cudaDeviceSynchronize());
    std::lock_guard<std::mutex> lk(g_mu);
    for (auto it = g_scratch.begin(); it != g_scratch.end();) {
        if (it->first.first == dev) {
            if (it->second.ptr) cudaFree(it->second.ptr);
            it = g_scratch.erase(it);
        } else ++it;
    }
    for (auto it = g_staging.begin(); it != g_staging.end();) {
        if (it->first.first == dev) {
            if (it->second.ptr) cudaFree(it->second.ptr);
            it = g_staging.erase(it);
        } else ++it;
    }
    auto pit = g_pipes.find(dev);  // copy streams / events of the pipelined _host entry points
    if (pit != g_pipes.end()) {
        HostPipe& p = pit->second;
        for (cudaEvent_t e : p.in_done) cudaEventDestroy(e);
        for (cudaEvent_t e : p.k_done) cudaEventDestroy(e);
        if (p.start) cudaEventDestroy(p.start);
        if (p.in) cudaStreamDestroy(p.in);
        if (p.out) cudaStreamDestroy(p.out);
        g_pipes.erase(pit);
    }
    return AFFINESCAN_OK;
}

}  // extern "C"
