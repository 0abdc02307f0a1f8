// affinescan_api.cu — C-ABI boundary of libaffinescan (include/affinescan.h): the exported
// entry points, error plumbing, the library-owned stream-ordered scratch, and the `_host`
// entry points (H2D || kernel || D2H pipelines).  No torch types, no exceptions.
#include <atomic>
#include <cstdint>
#include <limits>
#include <map>
#include <memory>
#include <mutex>
#include <tuple>
#include <utility>
#include <vector>

#include "host_internal.h"

namespace affinescan_host {

namespace {

thread_local int tl_last_cuda_error = 0;
thread_local int tl_last_variant = 0;
std::atomic<int64_t> g_launches{0};
std::atomic<int> g_opt_deterministic{0};

std::mutex g_mu;  // guards the maps below (never held across a device wait)

// ---------------------------------------------------------------- stream-ordered scratch
struct Buffer {
    void* ptr = nullptr;
    size_t bytes = 0;
    cudaEvent_t last_use = nullptr;  // recorded by scratch_release after the last launch
    uint64_t tick = 0;               // LRU clock
};
using ScratchKey = std::tuple<int, unsigned long long, int>;  // (device, stream id, slot)
std::map<ScratchKey, Buffer> g_scratch;
uint64_t g_scratch_tick = 0;

std::map<int, int> g_sm_count;

}  // namespace

int cuda_fail(cudaError_t e)
{
    tl_last_cuda_error = static_cast<int>(e);
    (void)cudaGetLastError();  // clear the sticky-less error state
    return AFFINESCAN_ERR_CUDA;
}

int after_launch()
{
    g_launches.fetch_add(1, std::memory_order_relaxed);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? AFFINESCAN_OK : cuda_fail(e);
}

void set_last_variant(int v) { tl_last_variant = v; }
bool deterministic_auto() { return g_opt_deterministic.load(std::memory_order_relaxed) != 0; }

int sm_count(int* out)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_sm_count.find(dev);
    if (it == g_sm_count.end()) {
        int n = 0;
        AS_CUDA(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev));
        it = g_sm_count.emplace(dev, n > 0 ? n : 1).first;
    }
    *out = it->second;
    return AFFINESCAN_OK;
}

namespace {
std::mutex g_attr_mu;
std::map<std::pair<const void*, int>, int> g_attr_done;
}  // namespace

int allow_dynamic_smem(const void* kernel, int bytes)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    const std::pair<const void*, int> key{kernel, dev};
    std::lock_guard<std::mutex> lk(g_attr_mu);
    auto it = g_attr_done.find(key);
    if (it == g_attr_done.end() || it->second < bytes) {
        AS_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
        g_attr_done[key] = bytes;
    }
    return AFFINESCAN_OK;
}

namespace {

// Frees the least recently used cached buffers of `dev` (never `keep`) until at most
// kScratchMaxEntries remain.  The free is enqueued on the CALLER's stream behind the buffer's
// last-use event, so it is safe whether or not the buffer's own stream still exists.
// g_mu is held.
int scratch_evict_lru(int dev, const ScratchKey& keep, cudaStream_t stream)
{
    while (true) {
        int count = 0;
        auto victim = g_scratch.end();
        for (auto it = g_scratch.begin(); it != g_scratch.end(); ++it) {
            if (std::get<0>(it->first) != dev) continue;
            ++count;
            if (it->first == keep) continue;
            if (victim == g_scratch.end() || it->second.tick < victim->second.tick) victim = it;
        }
        if (count <= kScratchMaxEntries || victim == g_scratch.end()) return AFFINESCAN_OK;
        Buffer b = victim->second;
        g_scratch.erase(victim);
        if (b.last_use) {
            AS_CUDA(cudaStreamWaitEvent(stream, b.last_use, 0));
            AS_CUDA(cudaEventDestroy(b.last_use));  // released once the wait has completed
        }
        if (b.ptr) AS_CUDA(cudaFreeAsync(b.ptr, stream));
    }
}

}  // namespace

int scratch_acquire(cudaStream_t stream, int slot, size_t bytes, Scratch* out)
{
    *out = Scratch{};
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    AS_CUDA(cudaStreamIsCapturing(stream, &cap));
    if (cap != cudaStreamCaptureStatusNone) {
        // inside a capture: the graph owns its scratch (alloc / memset / free nodes)
        AS_CUDA(cudaMallocAsync(&out->ptr, bytes, stream));
        AS_CUDA(cudaMemsetAsync(out->ptr, 0, bytes, stream));
        out->temporary = true;
        out->fresh = true;
        return AFFINESCAN_OK;
    }
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    unsigned long long sid = 0;
    AS_CUDA(cudaStreamGetId(stream, &sid));
    const ScratchKey key{dev, sid, slot};
    std::lock_guard<std::mutex> lk(g_mu);
    const bool is_new = g_scratch.find(key) == g_scratch.end();
    Buffer& b = g_scratch[key];
    b.tick = ++g_scratch_tick;
    if (is_new) AS_TRY(scratch_evict_lru(dev, key, stream));
    if (b.bytes < bytes) {
        // grow in stream order: earlier calls on this stream that still use the old buffer
        // finish before the free takes effect; nothing synchronises the host
        if (b.ptr) AS_CUDA(cudaFreeAsync(b.ptr, stream));
        b.ptr = nullptr;
        b.bytes = 0;
        const size_t want = bytes + bytes / 4 + 256;
        AS_CUDA(cudaMallocAsync(&b.ptr, want, stream));
        AS_CUDA(cudaMemsetAsync(b.ptr, 0, want, stream));
        b.bytes = want;
        out->fresh = true;
    }
    out->ptr = b.ptr;
    out->device = dev;
    out->stream_id = sid;
    out->slot = slot;
    return AFFINESCAN_OK;
}

int workspace_acquire(cudaStream_t stream, size_t bytes, Scratch* out)
{
    *out = Scratch{};
    AS_CUDA(cudaMallocAsync(&out->ptr, bytes > 0 ? bytes : 1, stream));
    out->temporary = true;
    out->fresh = true;
    return AFFINESCAN_OK;
}

int scratch_release(cudaStream_t stream, const Scratch& s)
{
    if (!s.ptr) return AFFINESCAN_OK;
    if (s.temporary) {
        AS_CUDA(cudaFreeAsync(s.ptr, stream));
        return AFFINESCAN_OK;
    }
    // cached buffer: remember where its last use ends, for a later eviction from another stream
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_scratch.find(ScratchKey{s.device, s.stream_id, s.slot});
    if (it == g_scratch.end() || it->second.ptr != s.ptr) return AFFINESCAN_OK;  // already evicted
    if (!it->second.last_use)
        AS_CUDA(cudaEventCreateWithFlags(&it->second.last_use, cudaEventDisableTiming));
    AS_CUDA(cudaEventRecord(it->second.last_use, stream));
    return AFFINESCAN_OK;
}

int scratch_cached_entries(int device)
{
    std::lock_guard<std::mutex> lk(g_mu);
    int n = 0;
    for (const auto& kv : g_scratch) n += std::get<0>(kv.first) == device;
    return n;
}

namespace {

// ---------------------------------------------------------------- host-buffer pipelines
// One context per (device, stream): its own staging buffers, copy streams and events, and its
// own mutex, so `_host` calls on different streams run concurrently and calls on the same
// stream serialise.  Staging grows with plain cudaMalloc AFTER synchronising the context's own
// streams (the `_host` entry points are synchronous by contract).
struct HostCtx {
    std::mutex mu;
    cudaStream_t in = nullptr, out = nullptr;
    cudaEvent_t start = nullptr;
    std::vector<cudaEvent_t> in_done, k_done;
    std::map<int, Buffer> staging;
};
std::map<std::pair<int, void*>, std::shared_ptr<HostCtx>> g_host;

int get_host_ctx(cudaStream_t stream, std::shared_ptr<HostCtx>* out)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_mu);
    auto& p = g_host[{dev, static_cast<void*>(stream)}];
    if (!p) p = std::make_shared<HostCtx>();
    *out = p;
    return AFFINESCAN_OK;
}

int ctx_streams(HostCtx& c, int nchunks)
{
    if (!c.in) {
        AS_CUDA(cudaStreamCreateWithFlags(&c.in, cudaStreamNonBlocking));
        AS_CUDA(cudaStreamCreateWithFlags(&c.out, cudaStreamNonBlocking));
        AS_CUDA(cudaEventCreateWithFlags(&c.start, cudaEventDisableTiming));
    }
    while (static_cast<int>(c.in_done.size()) < nchunks) {
        cudaEvent_t a = nullptr, b = nullptr;
        AS_CUDA(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
        AS_CUDA(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
        c.in_done.push_back(a);
        c.k_done.push_back(b);
    }
    return AFFINESCAN_OK;
}

int ctx_staging(HostCtx& c, cudaStream_t stream, int slot, size_t bytes, void** out)
{
    Buffer& b = c.staging[slot];
    if (bytes == 0) bytes = 1;
    if (b.bytes < bytes) {
        if (b.ptr) {
            // a previous call on this context has been synchronised before it returned
            AS_CUDA(cudaFree(b.ptr));
            b.ptr = nullptr;
            b.bytes = 0;
        }
        const size_t want = bytes + bytes / 4 + 256;
        AS_CUDA(cudaMalloc(&b.ptr, want));
        b.bytes = want;
    }
    (void)stream;
    *out = b.ptr;
    return AFFINESCAN_OK;
}

int ctx_stage_in(HostCtx& c, cudaStream_t stream, int slot, const void* host, size_t bytes,
                 void** dev)
{
    *dev = nullptr;
    if (!host) return AFFINESCAN_OK;
    AS_TRY(ctx_staging(c, stream, slot, bytes, dev));
    if (bytes) AS_CUDA(cudaMemcpyAsync(*dev, host, bytes, cudaMemcpyHostToDevice, stream));
    return AFFINESCAN_OK;
}

// After an error inside a pipelined `_host` call: drain everything this call enqueued, so no
// async copy into the caller's buffers is still in flight when the call returns.
void ctx_drain(HostCtx& c, cudaStream_t stream)
{
    if (c.in) (void)cudaStreamSynchronize(c.in);
    if (c.out) (void)cudaStreamSynchronize(c.out);
    (void)cudaStreamSynchronize(stream);
    (void)cudaGetLastError();
}

inline void* at(const void* p, size_t bytes)
{
    return const_cast<void*>(
        static_cast<const void*>(static_cast<const unsigned char*>(p) + bytes));
}

int affine_scan_host_locked(HostCtx& c, const void* a, const void* u, const float* h0, void* h,
                            float* h_last, int64_t num_seq, int64_t L, int io_dtype,
                            int64_t total, cudaStream_t stream)
{
    const size_t eb = static_cast<size_t>(total) * elt_size(io_dtype);
    const size_t sb = static_cast<size_t>(num_seq) * sizeof(float);
    void *da, *du, *dh0, *dh, *dhl = nullptr;
    AS_TRY(ctx_staging(c, stream, 0, eb, &da));
    AS_TRY(ctx_staging(c, stream, 1, eb, &du));
    AS_TRY(ctx_stage_in(c, stream, 2, h0, sb, &dh0));
    AS_TRY(ctx_staging(c, stream, 3, eb, &dh));
    if (h_last) AS_TRY(ctx_staging(c, stream, 4, sb, &dhl));
    if (total == 0) {  // nothing to scan: h_last <- h0 (or 0)
        AS_TRY(affine_scan_impl(da, du, static_cast<const float*>(dh0), dh,
                                static_cast<float*>(dhl), num_seq, L, io_dtype,
                                AFFINESCAN_VARIANT_AUTO, stream));
        if (h_last && sb) AS_CUDA(cudaMemcpyAsync(h_last, dhl, sb, cudaMemcpyDeviceToHost, stream));
        AS_CUDA(cudaStreamSynchronize(stream));
        return AFFINESCAN_OK;
    }
    // three-stage pipeline over chunks of whole sequences: H2D of chunk c+1 (copy-in stream) ||
    // kernel of chunk c (caller's stream) || D2H of chunk c-1 (copy-out stream)
    const size_t seq_bytes = static_cast<size_t>(L) * elt_size(io_dtype);
    int64_t per = static_cast<int64_t>((16u << 20) / seq_bytes) + 1;  // sequences per chunk
    if (per > num_seq) per = num_seq;
    int64_t nchunks = (num_seq + per - 1) / per;
    if (nchunks > 64) {  // bound the number of events
        nchunks = 64;
        per = (num_seq + nchunks - 1) / nchunks;
        nchunks = (num_seq + per - 1) / per;
    }
    AS_TRY(ctx_streams(c, static_cast<int>(nchunks)));
    AS_CUDA(cudaEventRecord(c.start, stream));
    AS_CUDA(cudaStreamWaitEvent(c.in, c.start, 0));
    AS_CUDA(cudaStreamWaitEvent(c.out, c.start, 0));
    for (int64_t k = 0; k < nchunks; ++k) {
        const int64_t s0 = k * per;
        const int64_t ns = (s0 + per <= num_seq) ? per : num_seq - s0;
        const size_t eo = seq_bytes * s0, so = sizeof(float) * s0;
        AS_CUDA(cudaMemcpyAsync(at(da, eo), at(a, eo), seq_bytes * ns, cudaMemcpyHostToDevice, c.in));
        AS_CUDA(cudaMemcpyAsync(at(du, eo), at(u, eo), seq_bytes * ns, cudaMemcpyHostToDevice, c.in));
        AS_CUDA(cudaEventRecord(c.in_done[k], c.in));
        AS_CUDA(cudaStreamWaitEvent(stream, c.in_done[k], 0));
        AS_TRY(affine_scan_impl(at(da, eo), at(du, eo),
                                dh0 ? static_cast<const float*>(at(dh0, so)) : nullptr, at(dh, eo),
                                dhl ? static_cast<float*>(at(dhl, so)) : nullptr, ns, L, io_dtype,
                                AFFINESCAN_VARIANT_AUTO, stream));
        AS_CUDA(cudaEventRecord(c.k_done[k], stream));
        AS_CUDA(cudaStreamWaitEvent(c.out, c.k_done[k], 0));
        AS_CUDA(cudaMemcpyAsync(at(h, eo), at(dh, eo), seq_bytes * ns, cudaMemcpyDeviceToHost, c.out));
        if (h_last)
            AS_CUDA(cudaMemcpyAsync(at(h_last, so), at(dhl, so), sizeof(float) * ns,
                                    cudaMemcpyDeviceToHost, c.out));
    }
    AS_CUDA(cudaStreamSynchronize(c.out));
    AS_CUDA(cudaStreamSynchronize(stream));
    return AFFINESCAN_OK;
}

int selective_host_locked(HostCtx& c, const SelectiveArgs& h, int64_t rows, int64_t total,
                          int64_t bnl, cudaStream_t stream)
{
    const size_t es = elt_size(h.io_dtype);
    const size_t xb = static_cast<size_t>(total) * es;
    const size_t bb = static_cast<size_t>(bnl) * es;
    const size_t ab = static_cast<size_t>(h.d_inner) * h.N * sizeof(float);
    const size_t db = static_cast<size_t>(h.d_inner) * sizeof(float);
    const size_t hb = static_cast<size_t>(rows) * h.N * sizeof(float);
    const size_t rb = static_cast<size_t>(h.batch) * static_cast<size_t>(h.L);
    void *dx, *dd, *dA, *dB, *dC, *dD, *dz = nullptr, *dbias, *drst = nullptr, *dh0, *dy,
         *dhl = nullptr;
    // Device staging (cached, full size), then a three-stage pipeline over batches:
    // H2D of batch b+1 (copy-in stream) || kernel of batch b (caller's stream) || D2H of batch
    // b-1 (copy-out stream).  PCIe is full duplex, so the step costs ~max(H2D, D2H), not the sum.
    AS_TRY(ctx_staging(c, stream, 10, xb, &dx));
    AS_TRY(ctx_staging(c, stream, 11, xb, &dd));
    AS_TRY(ctx_stage_in(c, stream, 12, h.A, ab, &dA));
    AS_TRY(ctx_staging(c, stream, 13, bb, &dB));
    AS_TRY(ctx_staging(c, stream, 14, bb, &dC));
    AS_TRY(ctx_stage_in(c, stream, 15, h.D, db, &dD));
    AS_TRY(ctx_stage_in(c, stream, 16, h.h0, hb, &dh0));
    AS_TRY(ctx_staging(c, stream, 17, xb, &dy));
    if (h.h_last) AS_TRY(ctx_staging(c, stream, 18, hb, &dhl));
    if (h.z) AS_TRY(ctx_staging(c, stream, 19, xb, &dz));
    AS_TRY(ctx_stage_in(c, stream, 20, h.delta_bias, db, &dbias));
    if (h.reset) AS_TRY(ctx_staging(c, stream, 21, rb, &drst));
    SelectiveArgs d = h;  // device-side view of one chunk
    d.A = static_cast<const float*>(dA);
    d.D = static_cast<const float*>(dD);
    d.delta_bias = static_cast<const float*>(dbias);
    d.variant = AFFINESCAN_VARIANT_AUTO;
    if (total == 0) {  // L == 0 (rows > 0): h_last <- h0 (or 0), as the device entry point does
        d.x = dx; d.delta = dd; d.B = dB; d.C = dC; d.y = dy; d.z = nullptr; d.reset = nullptr;
        d.h0 = static_cast<const float*>(dh0);
        d.h_last = static_cast<float*>(dhl);
        AS_TRY(selective_scan_impl(d, stream));
        if (h.h_last && hb) AS_CUDA(cudaMemcpyAsync(h.h_last, dhl, hb, cudaMemcpyDeviceToHost, stream));
        AS_CUDA(cudaStreamSynchronize(stream));
        return AFFINESCAN_OK;
    }
    // batches per chunk: at least ~16 MB of x per chunk so that copies stay at full PCIe rate
    const size_t xb1 = xb / h.batch, bb1 = bb / h.batch, hb1 = hb / h.batch, rb1 = rb / h.batch;
    int per = static_cast<int>((16u << 20) / (xb1 ? xb1 : 1)) + 1;
    if (per > h.batch) per = h.batch;
    const int nchunks = (h.batch + per - 1) / per;
    AS_TRY(ctx_streams(c, nchunks));
    // the small per-call tensors (A, D, bias, h0) went in on the caller's stream: the copy
    // streams must not overtake an earlier call's use of the staging buffers either
    AS_CUDA(cudaEventRecord(c.start, stream));
    AS_CUDA(cudaStreamWaitEvent(c.in, c.start, 0));
    AS_CUDA(cudaStreamWaitEvent(c.out, c.start, 0));
    for (int k = 0; k < nchunks; ++k) {
        const int b0 = k * per;
        const int nb = (b0 + per <= h.batch) ? per : h.batch - b0;
        const size_t xo = xb1 * b0, bo = bb1 * b0, ho = hb1 * b0, ro = rb1 * b0;
        AS_CUDA(cudaMemcpyAsync(at(dx, xo), at(h.x, xo), xb1 * nb, cudaMemcpyHostToDevice, c.in));
        AS_CUDA(cudaMemcpyAsync(at(dd, xo), at(h.delta, xo), xb1 * nb, cudaMemcpyHostToDevice, c.in));
        AS_CUDA(cudaMemcpyAsync(at(dB, bo), at(h.B, bo), bb1 * nb, cudaMemcpyHostToDevice, c.in));
        AS_CUDA(cudaMemcpyAsync(at(dC, bo), at(h.C, bo), bb1 * nb, cudaMemcpyHostToDevice, c.in));
        if (h.z) AS_CUDA(cudaMemcpyAsync(at(dz, xo), at(h.z, xo), xb1 * nb, cudaMemcpyHostToDevice, c.in));
        if (h.reset)
            AS_CUDA(cudaMemcpyAsync(at(drst, ro), at(h.reset, ro), rb1 * nb, cudaMemcpyHostToDevice, c.in));
        AS_CUDA(cudaEventRecord(c.in_done[k], c.in));
        AS_CUDA(cudaStreamWaitEvent(stream, c.in_done[k], 0));
        d.x = at(dx, xo); d.delta = at(dd, xo); d.B = at(dB, bo); d.C = at(dC, bo);
        d.z = h.z ? at(dz, xo) : nullptr;
        d.reset = h.reset ? static_cast<const unsigned char*>(at(drst, ro)) : nullptr;
        d.h0 = dh0 ? static_cast<const float*>(at(dh0, ho)) : nullptr;
        d.y = at(dy, xo);
        d.h_last = dhl ? static_cast<float*>(at(dhl, ho)) : nullptr;
        d.batch = nb;
        AS_TRY(selective_scan_impl(d, stream));
        AS_CUDA(cudaEventRecord(c.k_done[k], stream));
        AS_CUDA(cudaStreamWaitEvent(c.out, c.k_done[k], 0));
        AS_CUDA(cudaMemcpyAsync(at(h.y, xo), at(dy, xo), xb1 * nb, cudaMemcpyDeviceToHost, c.out));
        if (h.h_last)
            AS_CUDA(cudaMemcpyAsync(at(h.h_last, ho), at(dhl, ho), hb1 * nb, cudaMemcpyDeviceToHost,
                                    c.out));
    }
    AS_CUDA(cudaStreamSynchronize(c.out));
    AS_CUDA(cudaStreamSynchronize(stream));
    return AFFINESCAN_OK;
}

int selective_host(const SelectiveArgs& h, void* cuda_stream)
{
    if (h.io_dtype != AFFINESCAN_F32 && h.io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (h.batch < 0 || h.d_inner < 0 || h.L < 0) return AFFINESCAN_ERR_SHAPE;
    if (h.N < 1 || h.N > AFFINESCAN_MAX_N) return AFFINESCAN_ERR_UNSUPPORTED;
    int64_t rows = 0, total = 0, bnl = 0;
    if (mul_overflows(h.batch, h.d_inner, &rows) || mul_overflows(rows, h.L, &total) ||
        mul_overflows(static_cast<int64_t>(h.batch) * h.N, h.L, &bnl) ||
        total > (std::numeric_limits<int64_t>::max() >> 3) ||
        bnl > (std::numeric_limits<int64_t>::max() >> 3))
        return AFFINESCAN_ERR_SHAPE;
    if (total > 0 && (!h.x || !h.delta || !h.A || !h.B || !h.C || !h.y)) return AFFINESCAN_ERR_NULL;
    if (rows == 0) return AFFINESCAN_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    std::shared_ptr<HostCtx> ctx;
    AS_TRY(get_host_ctx(stream, &ctx));
    std::lock_guard<std::mutex> lk(ctx->mu);
    const int st = selective_host_locked(*ctx, h, rows, total, bnl, stream);
    if (st != AFFINESCAN_OK) ctx_drain(*ctx, stream);
    return st;
}

__global__ void reset_mask_from_cu_seqlens_kernel(const int* __restrict__ cu_seqlens, int num_seq,
                                                  unsigned char* __restrict__ reset, long long L)
{
    const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < num_seq) {
        const long long t = cu_seqlens[i];
        if (t >= 0 && t < L) reset[t] = 1;
    }
}

}  // namespace
}  // namespace affinescan_host

// =================================================================== exported C ABI
using namespace affinescan_host;

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
    if (num_seq == 0) return AFFINESCAN_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    std::shared_ptr<HostCtx> ctx;
    AS_TRY(get_host_ctx(stream, &ctx));
    std::lock_guard<std::mutex> lk(ctx->mu);
    const int st = affine_scan_host_locked(*ctx, a, u, h0, h, h_last, num_seq, L, io_dtype, total,
                                           stream);
    if (st != AFFINESCAN_OK) ctx_drain(*ctx, stream);
    return st;
}

static SelectiveArgs base_args(const void* x, const void* delta, const float* A, const void* B,
                               const void* C, const float* D, const float* h0, void* y,
                               float* h_last, int batch, int d_inner, int N, int64_t L,
                               int io_dtype, int variant)
{
    SelectiveArgs a;
    a.x = x; a.delta = delta; a.A = A; a.B = B; a.C = C; a.D = D; a.h0 = h0; a.y = y;
    a.h_last = h_last; a.batch = batch; a.d_inner = d_inner; a.N = N; a.L = L;
    a.io_dtype = io_dtype; a.variant = variant;
    return a;
}

int selective_scan_fwd(const void* x, const void* delta, const float* A, const void* B,
                       const void* C, const float* D, const float* h0, void* y, float* h_last,
                       int batch, int d_inner, int N, int64_t L, int io_dtype, void* cuda_stream)
{
    return selective_scan_impl(base_args(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N, L,
                                         io_dtype, AFFINESCAN_VARIANT_AUTO), cuda_stream);
}

int selective_scan_fwd_ex(const void* x, const void* delta, const float* A, const void* B,
                          const void* C, const float* D, const float* h0, void* y, float* h_last,
                          int batch, int d_inner, int N, int64_t L, int io_dtype, int variant,
                          void* cuda_stream)
{
    return selective_scan_impl(base_args(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N, L,
                                         io_dtype, variant), cuda_stream);
}

int selective_scan_fwd_host(const void* x, const void* delta, const float* A, const void* B,
                            const void* C, const float* D, const float* h0, void* y, float* h_last,
                            int batch, int d_inner, int N, int64_t L, int io_dtype,
                            void* cuda_stream)
{
    return selective_host(base_args(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N, L,
                                    io_dtype, AFFINESCAN_VARIANT_AUTO), cuda_stream);
}

int selective_scan_fwd_ext(const void* x, const void* delta, const float* A, const void* B,
                           const void* C, const float* D, const void* z, const float* delta_bias,
                           const uint8_t* reset, const float* h0, void* y, float* h_last,
                           int batch, int d_inner, int N, int64_t L, int io_dtype,
                           int delta_softplus, int a_structure, int variant, void* cuda_stream)
{
    SelectiveArgs a = base_args(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N, L, io_dtype,
                                variant);
    a.z = z; a.delta_bias = delta_bias; a.reset = reset;
    a.delta_softplus = delta_softplus ? 1 : 0;
    a.a_structure = a_structure;
    return selective_scan_impl(a, cuda_stream);
}

int selective_scan_fwd_ext_host(const void* x, const void* delta, const float* A, const void* B,
                                const void* C, const float* D, const void* z,
                                const float* delta_bias, const uint8_t* reset, const float* h0,
                                void* y, float* h_last, int batch, int d_inner, int N, int64_t L,
                                int io_dtype, int delta_softplus, int a_structure,
                                void* cuda_stream)
{
    SelectiveArgs a = base_args(x, delta, A, B, C, D, h0, y, h_last, batch, d_inner, N, L, io_dtype,
                                AFFINESCAN_VARIANT_AUTO);
    a.z = z; a.delta_bias = delta_bias; a.reset = reset;
    a.delta_softplus = delta_softplus ? 1 : 0;
    a.a_structure = a_structure;
    if (a_structure < AFFINESCAN_A_GENERAL || a_structure > AFFINESCAN_A_POWERS)
        return AFFINESCAN_ERR_UNSUPPORTED;
    return selective_host(a, cuda_stream);
}

int selective_scan_fwd_gated(const void* x, const void* delta_raw, const float* delta_bias,
                             const float* A, const void* B, const void* C, const float* D,
                             const void* z, const float* h0, void* y, float* h_last, int batch,
                             int d_inner, int N, int64_t L, int io_dtype, void* cuda_stream)
{
    return selective_scan_fwd_ext(x, delta_raw, A, B, C, D, z, delta_bias, nullptr, h0, y, h_last,
                                  batch, d_inner, N, L, io_dtype, 1, AFFINESCAN_A_GENERAL,
                                  AFFINESCAN_VARIANT_AUTO, cuda_stream);
}

int selective_scan_slice_aggregate(const void* x, const void* delta, const float* A, const void* B,
                                   const void* C, float* P, float* U, int batch, int d_inner,
                                   int N, int64_t L, int io_dtype, void* cuda_stream)
{
    SelectiveArgs a = base_args(x, delta, A, B, C, nullptr, nullptr, nullptr, nullptr, batch,
                                d_inner, N, L, io_dtype, AFFINESCAN_VARIANT_AUTO);
    return slice_aggregate_impl(a, P, U, cuda_stream);
}

int affinescan_compose_carry(const float* P_all, const float* U_all, const float* h0, float* h_in,
                             int rank, int world, int64_t n, void* cuda_stream)
{
    return compose_carry_impl(P_all, U_all, h0, h_in, rank, world, n, cuda_stream);
}

int affinescan_reset_mask_from_cu_seqlens(const int32_t* cu_seqlens, int num_seq, uint8_t* reset,
                                          int64_t L, void* cuda_stream)
{
    if (num_seq < 0 || L < 0) return AFFINESCAN_ERR_SHAPE;
    if (L == 0) return AFFINESCAN_OK;
    if (!reset || (num_seq > 0 && !cu_seqlens)) return AFFINESCAN_ERR_NULL;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    AS_CUDA(cudaMemsetAsync(reset, 0, static_cast<size_t>(L), stream));
    if (num_seq == 0) return AFFINESCAN_OK;
    reset_mask_from_cu_seqlens_kernel<<<(num_seq + 255) / 256, 256, 0, stream>>>(cu_seqlens, num_seq,
                                                                                 reset, L);
    return after_launch();
}

const char* affinescan_status_string(int status)
{
    switch (status) {
    case AFFINESCAN_OK: return "ok";
    case AFFINESCAN_ERR_NULL: return "a required pointer is NULL";
    case AFFINESCAN_ERR_SHAPE: return "negative or overflowing shape";
    case AFFINESCAN_ERR_DTYPE: return "unknown io dtype";
    case AFFINESCAN_ERR_UNSUPPORTED: return "unsupported N, variant, option or shape for the forced variant";
    case AFFINESCAN_ERR_CUDA: return "CUDA runtime error (see affinescan_last_cuda_error)";
    case AFFINESCAN_ERR_TOO_LARGE:
        return "problem exceeds the fixed scratch of affine_scan_static_scratch (65535 tiles: use "
               "affine_scan) or the workspace given to selective_scan_bwd_ws";
    default: return "unknown status";
    }
}

int affinescan_last_cuda_error(void) { return tl_last_cuda_error; }
int affinescan_last_variant(void) { return tl_last_variant; }
int64_t affinescan_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
int affinescan_version(void) { return 300; }
int affinescan_cached_scratch_buffers(void)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return scratch_cached_entries(dev);
}

int affinescan_set_option(int key, int value)
{
    if (key == AFFINESCAN_OPT_DETERMINISTIC) {
        if (value < -1 || value > 1) return AFFINESCAN_ERR_UNSUPPORTED;
        g_opt_deterministic.store(value == 1 ? 1 : 0);
        return AFFINESCAN_OK;
    }
    return set_lane_row_option(key, value);
}

int affinescan_release_cache(void)
{
    int dev = 0;
    AS_CUDA(cudaGetDevice(&dev));
    AS_CUDA(cudaDeviceSynchronize());
    // take the contexts out of the map first, then lock each one: a `_host` call running on
    // another thread keeps its context alive (shared_ptr) and finishes undisturbed
    std::vector<std::shared_ptr<HostCtx>> ctxs;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        for (auto it = g_scratch.begin(); it != g_scratch.end();) {
            if (std::get<0>(it->first) == dev) {
                if (it->second.ptr) cudaFree(it->second.ptr);
                if (it->second.last_use) cudaEventDestroy(it->second.last_use);
                it = g_scratch.erase(it);
            } else ++it;
        }
        for (auto it = g_host.begin(); it != g_host.end();) {
            if (it->first.first == dev) {
                ctxs.push_back(it->second);
                it = g_host.erase(it);
            } else ++it;
        }
    }
    for (auto& c : ctxs) {
        std::lock_guard<std::mutex> lk(c->mu);
        for (auto& kv : c->staging)
            if (kv.second.ptr) cudaFree(kv.second.ptr);
        c->staging.clear();
        for (cudaEvent_t e : c->in_done) cudaEventDestroy(e);
        for (cudaEvent_t e : c->k_done) cudaEventDestroy(e);
        c->in_done.clear();
        c->k_done.clear();
        if (c->start) cudaEventDestroy(c->start);
        if (c->in) cudaStreamDestroy(c->in);
        if (c->out) cudaStreamDestroy(c->out);
        c->start = nullptr;
        c->in = c->out = nullptr;
    }
    (void)cudaGetLastError();
    return AFFINESCAN_OK;
}

}  // extern "C"
