// host_internal.h — declarations shared by the host-side translation units of libaffinescan
// (affinescan_api.cu, affinescan_affine.cu, affinescan_selective.cu, affinescan_bwd.cu).
// Not part of the public ABI (include/affinescan.h is).
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/affinescan.h"

namespace affinescan_host {

// ---- error plumbing: every CUDA failure becomes AFFINESCAN_ERR_CUDA + a per-thread code
int cuda_fail(cudaError_t e);
int after_launch();              // counts the launch; turns cudaGetLastError() into a status
void set_last_variant(int v);

#define AS_CUDA(call)                                                        \
    do {                                                                     \
        const cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return ::affinescan_host::cuda_fail(e__);    \
    } while (0)
#define AS_TRY(call)                                   \
    do {                                               \
        const int st__ = (call);                       \
        if (st__ != AFFINESCAN_OK) return st__;        \
    } while (0)

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline size_t elt_size(int io_dtype) { return io_dtype == AFFINESCAN_BF16 ? 2 : 4; }
inline bool mul_overflows(int64_t a, int64_t b, int64_t* out)
{
    return __builtin_mul_overflow(a, b, out);
}

// ---- device facts (queried once per device)
int sm_count(int* out);          // cudaDevAttrMultiProcessorCount of the current device

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per (kernel, device); keyed by the
// kernel's address.
int allow_dynamic_smem(const void* kernel, int bytes);

// ---- library-owned device scratch, stream-ordered.
// scratch_acquire — SMALL scratch (look-back descriptors).  Outside stream capture: one cached
// buffer per (device, stream id, slot) that only grows; growing frees the old buffer with
// cudaFreeAsync and allocates with cudaMallocAsync ON THE CALLER'S STREAM, so no entry point
// ever synchronises the device.  The key is cudaStreamGetId, unique for the life of the process,
// not the raw handle: a new stream that reuses a destroyed stream's handle value never inherits
// (and races on) that stream's buffer.  At most kScratchMaxEntries buffers are kept per device:
// beyond that the least recently used one is freed on the caller's stream, ordered after its
// last use by an event, so buffers of streams that no longer exist do not pile up.  `fresh`
// tells the caller that the memory is new (zero-filled here, stream-ordered).
// Inside stream capture: a per-call cudaMallocAsync, zero-filled, that the caller returns with
// scratch_release (captured as alloc/free nodes, so the graph owns its scratch).
// workspace_acquire — LARGE per-call workspace (the backward pass): always a per-call
// cudaMallocAsync, NOT zero-filled, returned to the pool by scratch_release in stream order, so
// the library never pins hundreds of MB behind the back of the caller's allocator.
struct Scratch {
    void* ptr = nullptr;
    bool temporary = false;
    bool fresh = false;
    int device = 0;
    unsigned long long stream_id = 0;
    int slot = 0;
};
constexpr int kScratchMaxEntries = 64;
int scratch_acquire(cudaStream_t stream, int slot, size_t bytes, Scratch* out);
int workspace_acquire(cudaStream_t stream, size_t bytes, Scratch* out);
// Call after the last launch that uses the scratch (records the last-use event / frees).
int scratch_release(cudaStream_t stream, const Scratch& s);
int scratch_cached_entries(int device);  // introspection for tests

// ---- kernels' entry points behind the C ABI (implemented in the other translation units)
int affine_scan_impl(const void* a, const void* u, const float* h0, void* h, float* h_last,
                     int64_t num_seq, int64_t L, int io_dtype, int variant, void* cuda_stream);

struct SelectiveArgs {
    const void* x = nullptr;
    const void* delta = nullptr;
    const float* A = nullptr;
    const void* B = nullptr;
    const void* C = nullptr;
    const float* D = nullptr;
    const void* z = nullptr;
    const float* delta_bias = nullptr;
    const unsigned char* reset = nullptr;
    const float* h0 = nullptr;
    void* y = nullptr;
    float* h_last = nullptr;
    int batch = 0, d_inner = 0, N = 0;
    int64_t L = 0;
    int io_dtype = 0;
    int delta_softplus = 0;
    int a_structure = 0;
    int variant = 0;
};
int selective_scan_impl(const SelectiveArgs& a, void* cuda_stream);

// L-sharded scan helpers
int slice_aggregate_impl(const SelectiveArgs& a, float* P, float* U, void* cuda_stream);
int compose_carry_impl(const float* P_all, const float* U_all, const float* h0, float* h_in,
                       int rank, int world, int64_t n, void* cuda_stream);

int fill_h_last(const float* h0, float* h_last, int64_t n, cudaStream_t stream);

int set_lane_row_option(int key, int value);
// AFFINESCAN_OPT_DETERMINISTIC: AUTO never picks a decoupled look-back schedule
bool deterministic_auto();

}  // namespace affinescan_host
