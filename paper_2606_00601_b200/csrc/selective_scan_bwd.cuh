// selective_scan_bwd.cuh — backward pass of selective_scan_fwd (include/affinescan.h; SURVEY
// §8f-3; the paper evaluates "forward selective-scan workloads" only).
//
// For loss = <dy, y> + <dh_last, h_last> the adjoint of h_t = a_t h_{t-1} + u_t (Eq.3) is
// the same affine recurrence run right to left, g_t = a_{t+1} g_{t+1} + C_t dy_t (the monoid of
// P:90 Eq.7 with the roles of earlier/later swapped), and with a_t = exp(Delta_t A),
// u_t = Delta_t B_t x_t:
//     dC_t[n] += dy_t h_t[n]  (sum over d)      dD[d]   += dy_t x_t
//     dx_t     = D dy_t + Delta_t sum_n g_t[n] B_t[n]
//     dB_t[n] += g_t[n] Delta_t x_t  (sum over d)
//     dDelta_t = sum_n g_t[n] (A[n] a_t[n] h_{t-1}[n] + B_t[n] x_t)
//     dA[d,n] += g_t[n] Delta_t a_t[n] h_{t-1}[n]         dh0[n] = a_0[n] g_0[n]
//
// Schedule (the lane_row layout of the forward): one lane per (b,d) row, all N = 16 states in
// registers, a warp = 32 consecutive d of one batch so B_t/C_t are warp-uniform and are staged
// per warp as an fp32 [TC][2][N] shared-memory tile.  h_{t-1} is needed by the reverse sweep, and
// dividing it out of h_t is forbidden (Q17), so:
//   phase 1  forward sweep; the state entering every chunk of CK = 8 timesteps is checkpointed
//            to library scratch (coalesced: [row group][chunk][n][lane]);
//   phase 2  chunks in reverse: recompute the chunk's 8 states into shared memory, then run the
//            adjoint recurrence over its timesteps right to left.
// dB/dC partial sums over the 32 rows of a warp are formed with a shuffle reduce-scatter and
// written to scratch [row group][t][2N]; a second kernel adds the row groups of a batch in a
// FIXED order (no value atomics: bitwise reproducible, Q14).  dA/dD per-row partials
// are added over the batch by a third, tiny kernel.
#pragma once

#include "selective_common.cuh"

namespace affinescan {

constexpr int kBwdN = 16;    // states (the tuned case; other N: AFFINESCAN_ERR_UNSUPPORTED)
constexpr int kBwdCK = 8;    // timesteps per checkpointed chunk
constexpr int kBwdTC = 32;   // timesteps per staged B/C tile
constexpr int kBwdWarps = 4; // warps per CTA (autonomous)
constexpr int kBwdSmemPerWarp = kBwdTC * 2 * kBwdN * 4 + kBwdCK * kBwdN * 32 * 4;  // bc + hs

// v[j] of every lane -> lane j ends with sum over lanes of v[j] (returned); 31 shuffles.
__device__ __forceinline__ float warp_reduce_scatter32(float (&v)[32], int lane)
{
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const bool upper = (lane & off) != 0;
#pragma unroll
        for (int i = 0; i < off; ++i) {
            const float send = upper ? v[i] : v[i + off];
            const float keep = upper ? v[i + off] : v[i];
            v[i] = keep + __shfl_xor_sync(kFullMask, send, off);
        }
    }
    return v[0];
}

template <typename T>
__device__ __forceinline__ float load_io(const T* p);
template <>
__device__ __forceinline__ float load_io<float>(const float* p) { return __ldg(p); }
template <>
__device__ __forceinline__ float load_io<__nv_bfloat16>(const __nv_bfloat16* p)
{
    return __uint_as_float(
        static_cast<uint32_t>(__ldg(reinterpret_cast<const unsigned short*>(p))) << 16);
}

template <typename T>
__global__ void __launch_bounds__(kBwdWarps * 32)
selective_scan_bwd_kernel(const T* __restrict__ x, const T* __restrict__ delta,
                          const float* __restrict__ A, const T* __restrict__ B,
                          const T* __restrict__ C, const float* __restrict__ D,
                          const float* __restrict__ h0, const T* __restrict__ dy,
                          const float* __restrict__ dh_last, float* __restrict__ dx,
                          float* __restrict__ ddelta, float* __restrict__ dh0,
                          float* __restrict__ ckpt,     // [row groups][chunks][N][32]
                          float* __restrict__ part,     // [row groups][L][2N]  (dB | dC partials)
                          float* __restrict__ dA_part,  // [batch][d_inner][N]
                          float* __restrict__ dD_part,  // [batch][d_inner]
                          int batch, int d_inner, long long L)
{
    constexpr int N = kBwdN, CK = kBwdCK, TC = kBwdTC;
    constexpr int VEC = Io<T>::kVec;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const long long rows = static_cast<long long>(batch) * d_inner;
    const long long rg = static_cast<long long>(blockIdx.x) * kBwdWarps + warp;  // row group
    if (rg * 32 >= rows) return;
    const long long row = rg * 32 + lane;
    const int b = static_cast<int>((rg * 32) / d_inner);  // d_inner % 32 == 0: uniform
    const int d = static_cast<int>(row - static_cast<long long>(b) * d_inner);

    float* bc = reinterpret_cast<float*>(smem_raw + static_cast<size_t>(warp) * kBwdSmemPerWarp);
    float* hs = bc + TC * 2 * N;  // [CK][N][32]

    float A2[N];
#pragma unroll
    for (int q = 0; q < N / 4; ++q) {
        const float4 av = __ldg(reinterpret_cast<const float4*>(A + static_cast<long long>(d) * N) + q);
        A2[4 * q + 0] = av.x * kLog2e; A2[4 * q + 1] = av.y * kLog2e;
        A2[4 * q + 2] = av.z * kLog2e; A2[4 * q + 3] = av.w * kLog2e;
    }
    const float Dd = D ? __ldg(D + d) : 0.0f;
    const T* xr = x + row * L;
    const T* dr = delta + row * L;
    const T* dyr = dy + row * L;
    const long long nchunks = L / CK;  // L % CK == 0 (checked by the host)
    const long long ntiles = (L + TC - 1) / TC;
    float* ck = ckpt + rg * nchunks * N * 32 + lane;

    // B/C tile [TC][2][N] (fp32) of timesteps [t0, t0 + TC): lane j stages row j of (B | C)
    auto stage_tile = [&](long long t0) {
        __syncwarp();
        const T* src = (lane < N ? B : C) + (static_cast<long long>(b) * N + (lane & (N - 1))) * L + t0;
#pragma unroll
        for (int c = 0; c < TC / VEC; ++c) {
            float v[VEC];
            if (t0 + c * VEC < L) {
                unpack128<T>(__ldg(reinterpret_cast<const uint4*>(src) + c), v);
            } else {
#pragma unroll
                for (int k = 0; k < VEC; ++k) v[k] = 0.0f;
            }
#pragma unroll
            for (int k = 0; k < VEC; ++k) bc[(c * VEC + k) * 2 * N + lane] = v[k];
        }
        __syncwarp();
    };
    // the CK timesteps of x, delta (and dy) of one chunk
    auto load_chunk = [&](const T* p, long long t, float (&v)[CK]) {
#pragma unroll
        for (int c = 0; c < CK / VEC; ++c) {
            float w[VEC];
            unpack128<T>(__ldcs(reinterpret_cast<const uint4*>(p + t) + c), w);
#pragma unroll
            for (int k = 0; k < VEC; ++k) v[c * VEC + k] = w[k];
        }
    };

    // ------------------------------------------------------------------ phase 1: forward sweep
    float h[N];
#pragma unroll
    for (int n = 0; n < N; ++n) h[n] = h0 ? __ldg(h0 + row * N + n) : 0.0f;
    for (long long tile = 0; tile < ntiles; ++tile) {
        const long long t0 = tile * TC;
        stage_tile(t0);
        for (int c = 0; c < TC / CK && t0 + c * CK < L; ++c) {
            const long long t = t0 + c * CK;
            float* cko = ck + (t / CK) * N * 32;
#pragma unroll
            for (int n = 0; n < N; ++n) cko[n * 32] = h[n];
            float xv[CK], dl[CK];
            load_chunk(xr, t, xv);
            load_chunk(dr, t, dl);
#pragma unroll
            for (int k = 0; k < CK; ++k) {
                const float dxk = dl[k] * xv[k];
                const float* bt = bc + (c * CK + k) * 2 * N;
#pragma unroll
                for (int n = 0; n < N; ++n)
                    h[n] = fmaf(ex2_approx(dl[k] * A2[n]), h[n], dxk * bt[n]);
            }
        }
    }

    // ------------------------------------------------------------------ phase 2: reverse sweep
    float g[N], dAacc[N];
    float dDacc = 0.0f;
#pragma unroll
    for (int n = 0; n < N; ++n) {
        g[n] = dh_last ? __ldg(dh_last + row * N + n) : 0.0f;
        dAacc[n] = 0.0f;
    }
    float* prow = part + rg * L * 2 * N;
    for (long long tile = ntiles - 1; tile >= 0; --tile) {
        const long long t0 = tile * TC;
        stage_tile(t0);
        for (int c = TC / CK - 1; c >= 0; --c) {
            const long long t = t0 + c * CK;
            if (t >= L) continue;
            float xv[CK], dl[CK], dyv[CK];
            load_chunk(xr, t, xv);
            load_chunk(dr, t, dl);
            load_chunk(dyr, t, dyv);
            // recompute h_t for the chunk's timesteps into shared memory; hst = h_{t-1}
            float hst[N];
            const float* cki = ck + (t / CK) * N * 32;
#pragma unroll
            for (int n = 0; n < N; ++n) hst[n] = cki[n * 32];
            {
                float hh[N];
#pragma unroll
                for (int n = 0; n < N; ++n) hh[n] = hst[n];
#pragma unroll
                for (int k = 0; k < CK; ++k) {
                    const float dxk = dl[k] * xv[k];
                    const float* bt = bc + (c * CK + k) * 2 * N;
#pragma unroll
                    for (int n = 0; n < N; ++n) {
                        hh[n] = fmaf(ex2_approx(dl[k] * A2[n]), hh[n], dxk * bt[n]);
                        hs[(k * N + n) * 32 + lane] = hh[n];
                    }
                }
            }
            // adjoint recurrence, right to left
#pragma unroll
            for (int k = CK - 1; k >= 0; --k) {
                const float* bt = bc + (c * CK + k) * 2 * N;
                const float dxk = dl[k] * xv[k];
                float red[32];  // dB partials [0, N), dC partials [N, 2N)
                float s1 = 0.0f, sA = 0.0f;
#pragma unroll
                for (int n = 0; n < N; ++n) {
                    const float hn = hs[(k * N + n) * 32 + lane];
                    const float hp = k > 0 ? hs[((k - 1) * N + n) * 32 + lane] : hst[n];
                    g[n] = fmaf(bt[N + n], dyv[k], g[n]);       // + C_t dy_t
                    red[N + n] = dyv[k] * hn;                   // dC
                    red[n] = g[n] * dxk;                        // dB
                    s1 = fmaf(g[n], bt[n], s1);                 // sum_n g B
                    const float ga = g[n] * ex2_approx(dl[k] * A2[n]);
                    const float t1 = ga * hp;                   // g a h_{t-1}
                    sA = fmaf(A2[n], t1, sA);
                    dAacc[n] = fmaf(dl[k], t1, dAacc[n]);
                    g[n] = ga;                                  // carried to step t-1
                }
                dDacc = fmaf(dyv[k], xv[k], dDacc);
                if (dx) dx[row * L + t + k] = fmaf(Dd, dyv[k], dl[k] * s1);
                if (ddelta) ddelta[row * L + t + k] = fmaf(sA, kLn2, xv[k] * s1);
                const float tot = warp_reduce_scatter32(red, lane);
                prow[(t + k) * 2 * N + lane] = tot;
            }
            __syncwarp();  // hs is rewritten by the next chunk
        }
    }
    if (dh0) {
#pragma unroll
        for (int n = 0; n < N; ++n) dh0[row * N + n] = g[n];
    }
#pragma unroll
    for (int q = 0; q < N / 4; ++q)
        reinterpret_cast<float4*>(dA_part + row * N)[q] =
            make_float4(dAacc[4 * q], dAacc[4 * q + 1], dAacc[4 * q + 2], dAacc[4 * q + 3]);
    dD_part[row] = dDacc;
}

// dB[b][n][t] = sum over the row groups of batch b (in order) of part[rg][t][n]; dC likewise
// with n + N.  One CTA = (b, 32 timesteps): reads are 128-byte rows, the [t][2N] -> [2N][t]
// transpose goes through shared memory.
__global__ void __launch_bounds__(1024)
selective_scan_bwd_reduce_bc_kernel(const float* __restrict__ part, float* __restrict__ dB,
                                    float* __restrict__ dC, int groups_per_batch, long long L)
{
    __shared__ float tile[32][33];
    const int j = threadIdx.x & 31;   // index in [0, 2N)
    const int tt = threadIdx.x >> 5;  // timestep in the tile
    const int b = blockIdx.y;
    const long long t = static_cast<long long>(blockIdx.x) * 32 + tt;
    float acc = 0.0f;
    if (t < L) {
        const float* p = part + (static_cast<long long>(b) * groups_per_batch * L + t) * 32 + j;
        for (int rgi = 0; rgi < groups_per_batch; ++rgi) acc += p[static_cast<long long>(rgi) * L * 32];
    }
    tile[tt][j] = acc;
    __syncthreads();
    // thread (row = tt as index j', col = j as timestep): coalesced along t
    const int jj = tt, t2 = j;
    const long long tg = static_cast<long long>(blockIdx.x) * 32 + t2;
    if (tg < L) {
        float* dst = jj < kBwdN ? dB : dC;
        if (dst) dst[(static_cast<long long>(b) * kBwdN + (jj & (kBwdN - 1))) * L + tg] = tile[t2][jj];
    }
}

// dA[d][n] = sum_b dA_part[b][d][n]; dD[d] = sum_b dD_part[b][d]  (fixed order)
__global__ void selective_scan_bwd_reduce_ad_kernel(const float* __restrict__ dA_part,
                                                    const float* __restrict__ dD_part,
                                                    float* __restrict__ dA, float* __restrict__ dD,
                                                    int batch, int d_inner)
{
    const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    const long long nA = static_cast<long long>(d_inner) * kBwdN;
    if (i < nA && dA) {
        float acc = 0.0f;
        for (int b = 0; b < batch; ++b) acc += dA_part[static_cast<long long>(b) * nA + i];
        dA[i] = acc;
    }
    if (i < d_inner && dD) {
        float acc = 0.0f;
        for (int b = 0; b < batch; ++b) acc += dD_part[static_cast<long long>(b) * d_inner + i];
        dD[i] = acc;
    }
}

}  // namespace affinescan
