// affinescan_bwd.cu — host launch layer of selective_scan_bwd (include/affinescan.h).
#include <limits>

#include "host_internal.h"
#include "selective_scan_bwd.cuh"

namespace affinescan_host {

using namespace affinescan;
using bf16 = __nv_bfloat16;

namespace {

struct BwdArgs {
    const void *x, *delta, *B, *C, *dy;
    const float *A, *D, *h0, *dh_last;
    float *dx, *ddelta, *dA, *dB, *dC, *dD, *dh0;
    int batch, d_inner, N;
    int64_t L;
};

__global__ void copy_or_zero_kernel(const float* __restrict__ src, float* __restrict__ dst,
                                    long long n)
{
    const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src ? src[i] : 0.0f;
}

int copy_or_zero(const float* src, float* dst, int64_t n, cudaStream_t stream)
{
    if (!dst || n <= 0) return AFFINESCAN_OK;
    if ((n + 255) / 256 > 0x7fffffffLL) return AFFINESCAN_ERR_UNSUPPORTED;
    copy_or_zero_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, stream>>>(src, dst, n);
    return after_launch();
}

// fp32 words of [ckpt | part | dA_part | dD_part] for a supported shape
struct BwdLayout {
    size_t n_ckpt, n_part, n_da, n_dd;
    size_t bytes() const { return (n_ckpt + n_part + n_da + n_dd) * sizeof(float); }
};
BwdLayout bwd_layout(int batch, int d_inner, int64_t L)
{
    const int64_t rows = static_cast<int64_t>(batch) * d_inner;
    const int64_t groups = rows / kBwdRW;
    const int64_t nchunks = L / kBwdCK;
    return BwdLayout{static_cast<size_t>(groups) * nchunks * kBwdN * kBwdRW,
                     static_cast<size_t>(groups) * L * 2 * kBwdN,
                     static_cast<size_t>(rows) * kBwdN, static_cast<size_t>(rows)};
}

template <typename T>
int bwd_launch(const BwdArgs& a, void* workspace, int64_t workspace_bytes, cudaStream_t stream)
{
    const int64_t rows = static_cast<int64_t>(a.batch) * a.d_inner;
    const int64_t groups = rows / kBwdRW;
    // workspace: [ckpt | part | dA_part | dD_part], all fp32, ~16 B per (b,d,t).  The caller's
    // buffer if one was given; otherwise taken from the stream-ordered pool for THIS call only and
    // handed back when the last kernel below is done.  Every word is written before it is read,
    // so it is never cleared.
    const BwdLayout lay = bwd_layout(a.batch, a.d_inner, a.L);
    const size_t n_ckpt = lay.n_ckpt, n_part = lay.n_part, n_da = lay.n_da;
    auto kern = selective_scan_bwd_kernel<T>;
    constexpr int smem = kBwdSmemPerWarp * kBwdWarps;
    AS_TRY(allow_dynamic_smem(reinterpret_cast<const void*>(kern), smem));
    const int64_t blocks = (groups + kBwdWarps - 1) / kBwdWarps;
    // every launch limit is checked before anything is allocated or enqueued
    if (blocks > 0x7fffffffLL || a.L / 32 + 1 > 0x7fffffffLL || a.batch > 65535)
        return AFFINESCAN_ERR_UNSUPPORTED;
    Scratch sc;
    if (workspace) {
        if (!aligned16(workspace) || workspace_bytes < 0 ||
            static_cast<size_t>(workspace_bytes) < lay.bytes())
            return AFFINESCAN_ERR_TOO_LARGE;
    } else {
        AS_TRY(workspace_acquire(stream, lay.bytes(), &sc));
    }
    float* ckpt = static_cast<float*>(workspace ? workspace : sc.ptr);
    float* part = ckpt + n_ckpt;
    float* dA_part = part + n_part;
    float* dD_part = dA_part + n_da;
    kern<<<static_cast<unsigned>(blocks), kBwdWarps * 32, smem, stream>>>(
        static_cast<const T*>(a.x), static_cast<const T*>(a.delta), a.A, static_cast<const T*>(a.B),
        static_cast<const T*>(a.C), a.D, a.h0, static_cast<const T*>(a.dy), a.dh_last, a.dx,
        a.ddelta, a.dh0, ckpt, part, dA_part, dD_part, a.batch, a.d_inner, a.L);
    int st = after_launch();
    if (st == AFFINESCAN_OK && (a.dB || a.dC)) {
        const dim3 grid(static_cast<unsigned>((a.L + 31) / 32), static_cast<unsigned>(a.batch));
        selective_scan_bwd_reduce_bc_kernel<<<grid, 1024, 0, stream>>>(part, a.dB, a.dC,
                                                                       a.d_inner / kBwdRW, a.L);
        st = after_launch();
    }
    if (st == AFFINESCAN_OK && (a.dA || a.dD)) {
        const int64_t n = static_cast<int64_t>(a.d_inner) * kBwdN;
        selective_scan_bwd_reduce_ad_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, stream>>>(
            dA_part, dD_part, a.dA, a.dD, a.batch, a.d_inner);
        st = after_launch();
    }
    const int st2 = scratch_release(stream, sc);
    return st != AFFINESCAN_OK ? st : st2;
}

}  // namespace
}  // namespace affinescan_host

using namespace affinescan_host;

namespace {

bool bwd_shape_supported(int batch, int d_inner, int N, int64_t L)
{
    return N == kBwdN && d_inner % 32 == 0 && L % kBwdCK == 0 && batch <= 65535;
}

int bwd_entry(const void* x, const void* delta, const float* A, const void* B, const void* C,
              const float* D, const float* h0, const void* dy, const float* dh_last, float* dx,
              float* ddelta, float* dA, float* dB, float* dC, float* dD, float* dh0, int batch,
              int d_inner, int N, int64_t L, int io_dtype, void* workspace, int64_t workspace_bytes,
              void* cuda_stream)
{
    set_last_variant(0);
    if (io_dtype != AFFINESCAN_F32 && io_dtype != AFFINESCAN_BF16) return AFFINESCAN_ERR_DTYPE;
    if (batch < 0 || d_inner < 0 || L < 0) return AFFINESCAN_ERR_SHAPE;
    if (N < 1 || N > AFFINESCAN_MAX_N) return AFFINESCAN_ERR_UNSUPPORTED;
    int64_t rows = 0, total = 0, bnl = 0;
    if (mul_overflows(batch, d_inner, &rows) || mul_overflows(rows, L, &total) ||
        mul_overflows(static_cast<int64_t>(batch) * N, L, &bnl) ||
        total > (std::numeric_limits<int64_t>::max() >> 4) ||
        bnl > (std::numeric_limits<int64_t>::max() >> 3))
        return AFFINESCAN_ERR_SHAPE;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (rows == 0) return AFFINESCAN_OK;
    if (L == 0) {  // y is empty: only h_last = h0 depends on the inputs
        AS_TRY(copy_or_zero(nullptr, dA, static_cast<int64_t>(d_inner) * N, stream));
        AS_TRY(copy_or_zero(nullptr, dD, d_inner, stream));
        return copy_or_zero(dh_last, dh0, rows * N, stream);
    }
    if (!x || !delta || !A || !B || !C || !dy) return AFFINESCAN_ERR_NULL;
    // the tuned layout only: N = 16, two lanes per row with 16 rows of one batch per warp,
    // 128-bit accesses along L, 8-step checkpoint chunks
    if (!bwd_shape_supported(batch, d_inner, N, L) || !aligned16(x) || !aligned16(delta) ||
        !aligned16(B) || !aligned16(C) || !aligned16(dy) || !aligned16(A) || !aligned16(dx) ||
        !aligned16(ddelta))
        return AFFINESCAN_ERR_UNSUPPORTED;
    const BwdArgs a{x, delta, B, C, dy, A, D, h0, dh_last, dx, ddelta, dA, dB, dC, dD, dh0,
                    batch, d_inner, N, L};
    return io_dtype == AFFINESCAN_F32 ? bwd_launch<float>(a, workspace, workspace_bytes, stream)
                                      : bwd_launch<bf16>(a, workspace, workspace_bytes, stream);
}

}  // namespace

extern "C" {

int selective_scan_bwd(const void* x, const void* delta, const float* A, const void* B,
                       const void* C, const float* D, const float* h0, const void* dy,
                       const float* dh_last, float* dx, float* ddelta, float* dA, float* dB,
                       float* dC, float* dD, float* dh0, int batch, int d_inner, int N, int64_t L,
                       int io_dtype, void* cuda_stream)
{
    return bwd_entry(x, delta, A, B, C, D, h0, dy, dh_last, dx, ddelta, dA, dB, dC, dD, dh0, batch,
                     d_inner, N, L, io_dtype, nullptr, 0, cuda_stream);
}

int selective_scan_bwd_ws(const void* x, const void* delta, const float* A, const void* B,
                          const void* C, const float* D, const float* h0, const void* dy,
                          const float* dh_last, float* dx, float* ddelta, float* dA, float* dB,
                          float* dC, float* dD, float* dh0, int batch, int d_inner, int N,
                          int64_t L, int io_dtype, void* workspace, int64_t workspace_bytes,
                          void* cuda_stream)
{
    return bwd_entry(x, delta, A, B, C, D, h0, dy, dh_last, dx, ddelta, dA, dB, dC, dD, dh0, batch,
                     d_inner, N, L, io_dtype, workspace, workspace_bytes, cuda_stream);
}

int64_t selective_scan_bwd_workspace_bytes(int batch, int d_inner, int N, int64_t L)
{
    if (batch <= 0 || d_inner <= 0 || L <= 0 || !bwd_shape_supported(batch, d_inner, N, L))
        return 0;
    int64_t rows = 0, total = 0;
    if (mul_overflows(batch, d_inner, &rows) || mul_overflows(rows, L, &total) ||
        total > (std::numeric_limits<int64_t>::max() >> 5))
        return 0;
    return static_cast<int64_t>(bwd_layout(batch, d_inner, L).bytes());
}

}  // extern "C"
