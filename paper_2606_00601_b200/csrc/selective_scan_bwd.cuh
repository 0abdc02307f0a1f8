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
// Schedule (the lane_row layout of the forward): G = 2 lanes per (b,d) row, 8 of the N = 16 states
// per lane in registers, a warp = 16 consecutive d of one batch so B_t/C_t are warp-uniform and are
// staged per warp as an fp32 [TC][2][N] shared-memory tile.  h_{t-1} is needed by the reverse
// sweep, and dividing it out of h_t is forbidden (Q17), so:
//   phase 1  forward sweep; the state entering every chunk of CK = 8 timesteps is checkpointed
//            to library scratch (coalesced: [row group][chunk][n][row]);
//   phase 2  chunks in reverse: recompute the chunk's 8 states into shared memory, then run the
//            adjoint recurrence over its timesteps right to left.
// The x / delta / dy words and the checkpoint of a chunk are fetched one chunk ahead of their use.
// Sums over the states of a row (dx, ddelta) cross the lane pair with one shuffle each; dx and
// ddelta leave as 128-bit stores of CK timesteps, one lane of the pair each.  dB/dC partial sums
// over the 16 rows of a warp are formed with a shuffle reduce-scatter and written to scratch
// [row group][t][2N]; a second kernel adds the row groups of a batch in a FIXED order (no value
// atomics: bitwise reproducible, Q14).  dA/dD per-row partials are added over the batch
// by a third, tiny kernel.
#pragma once

#include "selective_common.cuh"

namespace affinescan {

constexpr int kBwdN = 16;    // states (the tuned case; other N: AFFINESCAN_ERR_UNSUPPORTED)
constexpr int kBwdCK = 8;    // timesteps per checkpointed chunk
constexpr int kBwdTC = 32;   // timesteps per staged B/C tile
constexpr int kBwdWarps = 4; // warps per CTA (autonomous)
constexpr int kBwdG = 2;     // lanes per (b,d) row: 8 states per lane, 16 rows per warp
constexpr int kBwdRW = 32 / kBwdG;  // rows per warp = rows per row group
constexpr int kBwdNS = kBwdN / kBwdG;
// per warp: B/C tile fp32 [TC][2][N] + recomputed states [CK][NS][32]
constexpr int kBwdSmemPerWarp = kBwdTC * 2 * kBwdN * 4 + kBwdCK * kBwdNS * 32 * 4;

// Reduce-scatter over the lanes that hold the same state slice (lanes l with equal l % G):
// v[i] of those 32/G lanes -> the lane with (lane / G) == i ends with the sum of v[i]
// (returned).  CNT = 32/G values, CNT - 1 shuffles.
template <int CNT, int G>
__device__ __forceinline__ float warp_reduce_scatter(float (&v)[CNT], int lane)
{
#pragma unroll
    for (int off = CNT / 2; off >= 1; off >>= 1) {
        const bool upper = (lane & (off * G)) != 0;
#pragma unroll
        for (int i = 0; i < off; ++i) {
            const float send = upper ? v[i] : v[i + off];
            const float keep = upper ? v[i + off] : v[i];
            v[i] = keep + __shfl_xor_sync(kFullMask, send, off * G);
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

// CK consecutive fp32 values of one row, written with 128-bit stores
__device__ __forceinline__ void store_chunk(float* p, const float (&v)[kBwdCK])
{
#pragma unroll
    for (int c = 0; c < kBwdCK / 4; ++c)
        __stcs(reinterpret_cast<float4*>(p) + c,
               make_float4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]));
}

template <typename T>
__global__ void __launch_bounds__(kBwdWarps * 32, 3)
selective_scan_bwd_kernel(const T* __restrict__ x, const T* __restrict__ delta,
                          const float* __restrict__ A, const T* __restrict__ B,
                          const T* __restrict__ C, const float* __restrict__ D,
                          const float* __restrict__ h0, const T* __restrict__ dy,
                          const float* __restrict__ dh_last, float* __restrict__ dx,
                          float* __restrict__ ddelta, float* __restrict__ dh0,
                          float* __restrict__ ckpt,     // [row groups][chunks][N][RW]
                          float* __restrict__ part,     // [row groups][L][2N]  (dB | dC partials)
                          float* __restrict__ dA_part,  // [batch][d_inner][N]
                          float* __restrict__ dD_part,  // [batch][d_inner]
                          int batch, int d_inner, long long L)
{
    constexpr int N = kBwdN, CK = kBwdCK, TC = kBwdTC, G = kBwdG, RW = kBwdRW, NS = kBwdNS;
    constexpr int VEC = Io<T>::kVec;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int g = lane % G;   // which NS-slice of the row's states
    const int rl = lane / G;  // row within the warp's group
    const long long rows = static_cast<long long>(batch) * d_inner;
    const long long rg = static_cast<long long>(blockIdx.x) * kBwdWarps + warp;  // row group
    if (rg * RW >= rows) return;
    const long long row = rg * RW + rl;
    const int b = static_cast<int>((rg * RW) / d_inner);  // d_inner % 32 == 0: uniform
    const int d = static_cast<int>(row - static_cast<long long>(b) * d_inner);

    float* bc = reinterpret_cast<float*>(smem_raw + static_cast<size_t>(warp) * kBwdSmemPerWarp);
    float* hs = bc + TC * 2 * N;  // [CK][NS][32]

    float A2[NS];
#pragma unroll
    for (int q = 0; q < NS / 4; ++q) {
        const float4 av =
            __ldg(reinterpret_cast<const float4*>(A + static_cast<long long>(d) * N + g * NS) + q);
        A2[4 * q + 0] = av.x * kLog2e; A2[4 * q + 1] = av.y * kLog2e;
        A2[4 * q + 2] = av.z * kLog2e; A2[4 * q + 3] = av.w * kLog2e;
    }
    const float Dd = D ? __ldg(D + d) : 0.0f;
    const T* xr = x + row * L;
    const T* dr = delta + row * L;
    const T* dyr = dy + row * L;
    const long long nchunks = L / CK;  // L % CK == 0 (checked by the host)
    const long long ntiles = (L + TC - 1) / TC;
    // checkpoint of (chunk, state n, row rl): [rg][chunk][n][rl]
    float* ck = ckpt + rg * nchunks * N * RW + (g * NS) * RW + rl;

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
    // the CK timesteps of x, delta (and dy) of one chunk: raw 128-bit words, fetched one chunk
    // ahead of their use (a chunk is ~1.5 k instructions of arithmetic: enough to cover HBM)
    constexpr int QW = CK / VEC;  // 128-bit words per chunk and array
    struct Raw { uint4 w[QW]; };
    auto fetch = [&](const T* p, long long t) {
        Raw r;
#pragma unroll
        for (int c = 0; c < QW; ++c) r.w[c] = __ldcs(reinterpret_cast<const uint4*>(p + t) + c);
        return r;
    };
    auto widen = [&](const Raw& r, float (&v)[CK]) {
#pragma unroll
        for (int c = 0; c < QW; ++c) {
            float w[VEC];
            unpack128<T>(r.w[c], w);
#pragma unroll
            for (int k = 0; k < VEC; ++k) v[c * VEC + k] = w[k];
        }
    };

    // ------------------------------------------------------------------ phase 1: forward sweep
    float h[NS];
#pragma unroll
    for (int n = 0; n < NS; ++n) h[n] = h0 ? __ldg(h0 + row * N + g * NS + n) : 0.0f;
    Raw xq = fetch(xr, 0), dq = fetch(dr, 0);
    for (long long tile = 0; tile < ntiles; ++tile) {
        const long long t0 = tile * TC;
        stage_tile(t0);
        for (int c = 0; c < TC / CK && t0 + c * CK < L; ++c) {
            const long long t = t0 + c * CK;
            float* cko = ck + (t / CK) * N * RW;
#pragma unroll
            for (int n = 0; n < NS; ++n) cko[n * RW] = h[n];
            float xv[CK], dl[CK];
            widen(xq, xv);
            widen(dq, dl);
            {
                const long long tn = t + CK < L ? t + CK : t;  // past the end: re-read, unused
                xq = fetch(xr, tn);
                dq = fetch(dr, tn);
            }
#pragma unroll
            for (int k = 0; k < CK; ++k) {
                const float dxk = dl[k] * xv[k];
                const float* bt = bc + (c * CK + k) * 2 * N + g * NS;
#pragma unroll
                for (int n = 0; n < NS; ++n)
                    h[n] = fmaf(ex2_approx(dl[k] * A2[n]), h[n], dxk * bt[n]);
            }
        }
    }

    // ------------------------------------------------------------------ phase 2: reverse sweep
    float gv[NS], dAacc[NS];
    float dDacc = 0.0f;
#pragma unroll
    for (int n = 0; n < NS; ++n) {
        gv[n] = dh_last ? __ldg(dh_last + row * N + g * NS + n) : 0.0f;
        dAacc[n] = 0.0f;
    }
    float* prow = part + rg * L * 2 * N;
    // the value this lane ends the reduce-scatter with: index i = lane / G of its slice's
    // [dB(NS) | dC(NS)] vector -> position in the [2N] row of `part`
    const int pi = rl;                                          // 0 .. 2 NS - 1 (RW == 2 NS)
    const int pj = (pi < NS ? 0 : N) + g * NS + (pi & (NS - 1));
    static_assert(RW == 2 * NS, "one reduced value per lane");
    Raw yq;
    float hq[NS];  // checkpoint of the next chunk to be processed
    {
        const long long tl = L - CK;
        xq = fetch(xr, tl);
        dq = fetch(dr, tl);
        yq = fetch(dyr, tl);
        const float* cki = ck + (tl / CK) * N * RW;
#pragma unroll
        for (int n = 0; n < NS; ++n) hq[n] = cki[n * RW];
    }
    for (long long tile = ntiles - 1; tile >= 0; --tile) {
        const long long t0 = tile * TC;
        stage_tile(t0);
        for (int c = TC / CK - 1; c >= 0; --c) {
            const long long t = t0 + c * CK;
            if (t >= L) continue;
            float xv[CK], dl[CK], dyv[CK];
            widen(xq, xv);
            widen(dq, dl);
            widen(yq, dyv);
            // recompute h_t for the chunk's timesteps into shared memory; hst = h_{t-1}
            float hst[NS];
#pragma unroll
            for (int n = 0; n < NS; ++n) hst[n] = hq[n];
            {
                const long long tp = t >= CK ? t - CK : t;  // before the start: re-read, unused
                xq = fetch(xr, tp);
                dq = fetch(dr, tp);
                yq = fetch(dyr, tp);
                const float* cki = ck + (tp / CK) * N * RW;
#pragma unroll
                for (int n = 0; n < NS; ++n) hq[n] = cki[n * RW];
            }
            {
                float hh[NS];
#pragma unroll
                for (int n = 0; n < NS; ++n) hh[n] = hst[n];
#pragma unroll
                for (int k = 0; k < CK; ++k) {
                    const float dxk = dl[k] * xv[k];
                    const float* bt = bc + (c * CK + k) * 2 * N + g * NS;
#pragma unroll
                    for (int n = 0; n < NS; ++n) {
                        hh[n] = fmaf(ex2_approx(dl[k] * A2[n]), hh[n], dxk * bt[n]);
                        hs[(k * NS + n) * 32 + lane] = hh[n];
                    }
                }
            }
            // adjoint recurrence, right to left
            float dxo[CK], ddo[CK];
#pragma unroll
            for (int k = CK - 1; k >= 0; --k) {
                const float* bt = bc + (c * CK + k) * 2 * N + g * NS;
                const float dxk = dl[k] * xv[k];
                float red[2 * NS];  // dB partials [0, NS), dC partials [NS, 2 NS) of this slice
                float s1 = 0.0f, sA = 0.0f;
#pragma unroll
                for (int n = 0; n < NS; ++n) {
                    const float hn = hs[(k * NS + n) * 32 + lane];
                    const float hp = k > 0 ? hs[((k - 1) * NS + n) * 32 + lane] : hst[n];
                    gv[n] = fmaf(bt[N + n], dyv[k], gv[n]);     // + C_t dy_t
                    red[NS + n] = dyv[k] * hn;                  // dC
                    red[n] = gv[n] * dxk;                       // dB
                    s1 = fmaf(gv[n], bt[n], s1);                // sum_n g B
                    const float ga = gv[n] * ex2_approx(dl[k] * A2[n]);
                    const float t1 = ga * hp;                   // g a h_{t-1}
                    sA = fmaf(A2[n], t1, sA);
                    dAacc[n] = fmaf(dl[k], t1, dAacc[n]);
                    gv[n] = ga;                                 // carried to step t-1
                }
                // sums over the row's states: add the other slice's share
                s1 += __shfl_xor_sync(kFullMask, s1, 1);
                sA += __shfl_xor_sync(kFullMask, sA, 1);
                dDacc = fmaf(dyv[k], xv[k], dDacc);
                dxo[k] = fmaf(Dd, dyv[k], dl[k] * s1);
                ddo[k] = fmaf(sA, kLn2, xv[k] * s1);
                const float tot = warp_reduce_scatter<2 * NS, G>(red, lane);
                prow[(t + k) * 2 * N + pj] = tot;
            }
            // one lane of the row writes dx, the other ddelta: CK fp32 each, 128-bit stores
            if (g == 0) {
                if (dx) store_chunk(dx + row * L + t, dxo);
            } else {
                if (ddelta) store_chunk(ddelta + row * L + t, ddo);
            }
            __syncwarp();  // hs is rewritten by the next chunk
        }
    }
    if (dh0) {
#pragma unroll
        for (int n = 0; n < NS; ++n) dh0[row * N + g * NS + n] = gv[n];
    }
#pragma unroll
    for (int q = 0; q < NS / 4; ++q)
        reinterpret_cast<float4*>(dA_part + row * N + g * NS)[q] =
            make_float4(dAacc[4 * q], dAacc[4 * q + 1], dAacc[4 * q + 2], dAacc[4 * q + 3]);
    if (g == 0) dD_part[row] = dDacc;
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
