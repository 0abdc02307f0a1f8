// affinescan_static_scratch.cu — affine_scan_static_scratch (include/affinescan.h): the
// decoupled look-back scan of affine_scan for callers that are not allowed to allocate
// device memory.
//
// Who needs this.  The ordinary AFFINESCAN_AFFINE_LOOKBACK path keeps its tile descriptors in
// library scratch obtained with cudaMallocAsync (affinescan_api.cu::scratch_acquire).  Some
// hosts cannot live with that: a process whose whole device-memory budget was handed to another
// allocator at start-up (a serving engine that pre-sizes its KV cache to "everything that is
// left", a framework whose caching allocator must account for every byte), a real-time loop that
// may not take the driver's allocation lock or page-table work on its hot path, or a sandboxed
// plug-in that is given input and output buffers and nothing else.  For them the descriptors live
// in a fixed array that is part of the library image: it exists on every GPU from the moment the
// library's module is loaded there until the process exits, and this entry point never calls
// cudaMalloc, cudaMallocAsync, cudaFree or any library routine that allocates device memory.
//
// The price: a hard size limit (kStaticMaxTiles tiles), 1 MiB of device memory held per GPU
// whether or not the entry point is ever called, and ONE array shared by every call on a device,
// so two calls whose kernels overlap on the GPU (different streams, different host threads, a
// graph replayed beside a direct call) corrupt each other.  Serialise them.
#include <limits>
#include <mutex>

#include "affine_scan.cuh"
#include "host_internal.h"

namespace affinescan_host {

using namespace affinescan;
using bf16 = __nv_bfloat16;

namespace {

// Same tiling as the allocating path (affinescan_affine.cu) so both run the same kernels.
constexpr int kSsWarps = 8;
constexpr int kSsJ = 4;
constexpr int kSsStages = 3;
constexpr int kSsCtasPerSm = 2;

// [LookbackCtrl (16 B) | kStaticMaxTiles descriptors of 16 B] = exactly 1 MiB.
constexpr long long kStaticMaxTiles = 65535;
constexpr size_t kStaticWords = 2 + 2 * static_cast<size_t>(kStaticMaxTiles);  // 64-bit words
static_assert(sizeof(LookbackCtrl) == 16, "control block is two 64-bit words");
static_assert(kStaticWords * 8 == (1u << 20), "static scratch is 1 MiB");

// Zero-initialised when the module is loaded on a device.  In HOST code this name is only a
// handle for cudaGetSymbolAddress: it is not a device address and must never be passed to a
// kernel as one.
static __device__ __align__(256) unsigned long long g_static_scratch[kStaticWords];

constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_addr[kMaxDevices] = {};

// Device address of g_static_scratch on the CURRENT device, looked up once per device.
int static_scratch_address(void** out)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return AFFINESCAN_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_addr[dev]) {
        void* p = nullptr;
        AS_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return AFFINESCAN_ERR_CUDA;
        g_static_addr[dev] = p;
    }
    *out = g_static_addr[dev];
    return AFFINESCAN_OK;
}

template <typename T, int VEC>
constexpr long long static_tile_elems()
{
    return static_cast<long long>(kSsWarps) * 32 * VEC * kSsJ;
}

template <typename T, int VEC>
int launch_static(const T* a, const T* u, const float* h0, T* h, float* h_last, int64_t total,
                  int64_t L, cudaStream_t stream)
{
    constexpr long long kTile = static_tile_elems<T, VEC>();
    const int64_t ntiles = (total + kTile - 1) / kTile;
    if (ntiles > kStaticMaxTiles) return AFFINESCAN_ERR_TOO_LARGE;
    void* base = nullptr;
    AS_TRY(static_scratch_address(&base));
    auto* ctrl = static_cast<LookbackCtrl*>(base);
    auto* desc = reinterpret_cast<unsigned long long*>(ctrl + 1);
    // The array keeps whatever the previous call left.  The tile ticket and the count of
    // finished tiles must start at zero (a launch re-arms them when it ends, but a launch that
    // never finished would not have); the epoch word after them must SURVIVE: it is what makes
    // the descriptors of earlier calls read as empty, so they are not cleared.
    AS_CUDA(cudaMemsetAsync(ctrl, 0, 2 * sizeof(unsigned), stream));
    if constexpr (VEC > 1) {
        using S = ChainSmem<T, VEC, kSsJ, kSsWarps, kSsStages>;
        auto kern = affine_scan_chain_kernel<T, VEC, kSsJ, kSsWarps, kSsStages, kSsCtasPerSm>;
        AS_TRY(allow_dynamic_smem(reinterpret_cast<const void*>(kern), S::kBytes));
        int sms = 0;
        AS_TRY(sm_count(&sms));
        const int64_t resident = static_cast<int64_t>(sms) * kSsCtasPerSm;
        const unsigned grid = static_cast<unsigned>(ntiles < resident ? ntiles : resident);
        kern<<<grid, (kSsWarps + 1) * 32, S::kBytes, stream>>>(a, u, h0, h, h_last, total, L,
                                                               ntiles, desc, ctrl);
    } else {
        affine_scan_lookback_kernel<T, VEC, kSsJ, kSsWarps>
            <<<static_cast<unsigned>(ntiles), kSsWarps * 32, 0, stream>>>(a, u, h0, h, h_last,
                                                                          total, L, desc, ctrl);
    }
    return after_launch();
}

template <typename T>
int static_dispatch(const void* a_, const void* u_, const float* h0, void* h_, float* h_last,
                    int64_t total, int64_t L, cudaStream_t stream)
{
    const T* a = static_cast<const T*>(a_);
    const T* u = static_cast<const T*>(u_);
    T* h = static_cast<T*>(h_);
    constexpr int kVec = Io<T>::kVec;
    const bool vec_ok = (L % kVec == 0) && aligned16(a) && aligned16(u) && aligned16(h);
    return vec_ok ? launch_static<T, kVec>(a, u, h0, h, h_last, total, L, stream)
                  : launch_static<T, 1>(a, u, h0, h, h_last, total, L, stream);
}

}  // namespace

}  // namespace affinescan_host

using namespace affinescan_host;

extern "C" {

int64_t affine_scan_static_scratch_max_elements(int io_dtype, int vectorised)
{
    if (io_dtype != AFFINESCAN_F32 && io_dtype != AFFINESCAN_BF16) return 0;
    const long long tile =
        !vectorised ? static_tile_elems<float, 1>()
        : io_dtype == AFFINESCAN_F32 ? static_tile_elems<float, Io<float>::kVec>()
                                     : static_tile_elems<bf16, Io<bf16>::kVec>();
    return kStaticMaxTiles * tile;
}

int affine_scan_static_scratch(const void* a, const void* u, const float* h0, void* h,
                               float* h_last, int64_t num_seq, int64_t L, int io_dtype,
                               void* cuda_stream)
{
    set_last_variant(0);
    if (io_dtype != AFFINESCAN_F32 && io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (num_seq < 0 || L < 0) return AFFINESCAN_ERR_SHAPE;
    int64_t total = 0;
    if (mul_overflows(num_seq, L, &total) || total > (std::numeric_limits<int64_t>::max() >> 3))
        return AFFINESCAN_ERR_SHAPE;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (num_seq == 0) return AFFINESCAN_OK;
    if (L == 0) return fill_h_last(h0, h_last, num_seq, stream);  // no scratch involved
    // the size check comes before the pointer checks and before any device work, so a caller can
    // probe the limit without buffers
    const bool could_vectorise = L % (io_dtype == AFFINESCAN_F32 ? 4 : 8) == 0;
    if (total > affine_scan_static_scratch_max_elements(io_dtype, could_vectorise))
        return AFFINESCAN_ERR_TOO_LARGE;
    if (!a || !u || !h) return AFFINESCAN_ERR_NULL;
    const int st = io_dtype == AFFINESCAN_F32
                       ? static_dispatch<float>(a, u, h0, h, h_last, total, L, stream)
                       : static_dispatch<bf16>(a, u, h0, h, h_last, total, L, stream);
    if (st == AFFINESCAN_OK) set_last_variant(AFFINESCAN_AFFINE_LOOKBACK);
    return st;
}

}  // extern "C"
