/*
 * affinescan.h — C ABI of libaffinescan: the affine-pair associative scan of
 * arxiv/paper_2606_00601 ("ScanWeaver") and its main instance, the Mamba-style
 * fused selective-scan forward, as hand-written CUDA kernels for sm_100a (B200).
 *
 * Citations:  P:<n>  = line n of /root/reference/PAPER.md
 *             BJ     = BASELINE.json north_star / configs
 *             Q<k>   = reading k in DESIGN.md ("Readings of the paper")
 *
 * Conventions common to every entry point
 *   - Plain pointers and sizes only.  Unless the name ends in `_host`, every data
 *     pointer is a DEVICE pointer on the current CUDA device; `_host` entry points
 *     take HOST pointers (pinned or pageable) and do the copies themselves.
 *   - All tensors are dense, row-major, last index contiguous; no strides.
 *   - The caller owns every buffer.  Inputs are never written.  Outputs must not
 *     alias inputs (in-place is unsupported).
 *   - Device entry points are asynchronous on `cuda_stream` (a cudaStream_t cast to
 *     void*; NULL = the legacy default stream): they enqueue work and return without
 *     synchronising.  `_host` entry points synchronise `cuda_stream` before returning.
 *   - The library owns only a small per-(device, stream) scratch for the decoupled
 *     look-back tile descriptors.  It is allocated, grown and cleared IN STREAM ORDER on
 *     `cuda_stream` (cudaMallocAsync / cudaFreeAsync / cudaMemsetAsync): no device entry
 *     point synchronises the host or the device, and none clears the scratch per call
 *     (descriptor statuses carry a per-launch epoch).  At most 64 such buffers are kept per
 *     device (least recently used freed first, in stream order), keyed by the stream's id, so
 *     buffers of destroyed streams neither pile up nor get inherited by a stream that reuses
 *     the handle.  The large workspace of selective_scan_bwd is NOT cached: it is a per-call
 *     cudaMallocAsync / cudaFreeAsync on `cuda_stream` (memory goes back to the device's
 *     stream-ordered pool, where the caller's allocator policy decides what happens to it).
 *     affine_scan_static_scratch allocates nothing at all.  Device entry points may be captured
 *     in a CUDA graph: inside a capture the scratch is a per-call stream-ordered
 *     allocation owned by the graph.  A captured graph must not run concurrently with
 *     itself.  Calls on different streams may run concurrently from different threads.
 *   - Errors are integer status codes (affinescan_status); nothing aborts, throws or
 *     prints.  Misaligned pointers or an L that is not a multiple of the 128-bit
 *     vector width are NOT errors: a scalar-load kernel is chosen.
 *   - State and accumulation are fp32; io dtype is fp32 or bf16; outputs are rounded
 *     to the io dtype with round-to-nearest-even; h_last is always fp32.
 *   - Results are bitwise reproducible run to run for a given variant (values are
 *     never accumulated with atomics), except AFFINESCAN_AFFINE_LOOKBACK and
 *     AFFINESCAN_SELECTIVE_CHUNKED, whose decoupled look-back folds whichever predecessor
 *     aggregates are published at poll time: reproducible up to the floating-point
 *     association order of P:90 Eq.(7) (all orders are within the stated tolerance).
 *     AFFINESCAN_VARIANT_AUTO picks these two for one or few long sequences / few rows x long
 *     L; affinescan_set_option(AFFINESCAN_OPT_DETERMINISTIC, 1) keeps AUTO off them.
 */
#ifndef AFFINESCAN_H_
#define AFFINESCAN_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define AFFINESCAN_API
#else
#define AFFINESCAN_API __attribute__((visibility("default")))
#endif

typedef enum affinescan_status {
    AFFINESCAN_OK = 0,
    AFFINESCAN_ERR_NULL = 1,        /* a required pointer is NULL                         */
    AFFINESCAN_ERR_SHAPE = 2,       /* negative size, or a size product overflows int64   */
    AFFINESCAN_ERR_DTYPE = 3,       /* io_dtype is not an affinescan_dtype                */
    AFFINESCAN_ERR_UNSUPPORTED = 4, /* N outside [1, AFFINESCAN_MAX_N]; unknown variant;
                                       a forced variant that cannot run this shape        */
    AFFINESCAN_ERR_CUDA = 5,        /* a CUDA runtime call failed; see
                                       affinescan_last_cuda_error()                       */
    AFFINESCAN_ERR_TOO_LARGE = 6    /* the problem needs more scratch than the fixed array of
                                       affine_scan_static_scratch, or the workspace given
                                       to selective_scan_bwd_ws, holds                    */
} affinescan_status;

typedef enum affinescan_dtype {
    AFFINESCAN_F32 = 0,  /* IEEE binary32 */
    AFFINESCAN_BF16 = 1  /* bfloat16      */
} affinescan_dtype;

#define AFFINESCAN_MAX_N 64

/* Kernel variants.  AUTO picks from the shape; the others force one schedule (tests,
 * ablations, benchmarks). */
typedef enum affinescan_variant {
    AFFINESCAN_VARIANT_AUTO = 0,
    /* affine_scan */
    AFFINESCAN_AFFINE_LOOKBACK = 1, /* single pass over the flattened [num_seq*L] stream by
                                       persistent CTAs (tiles streamed through a TMA ring);
                                       decoupled look-back carry between tiles; sequence
                                       heads are reset pairs (0, a0*h0+u0)  (BJ)          */
    AFFINESCAN_AFFINE_CTA_LOOP = 2, /* one CTA per sequence, loop over L with the carry in
                                       a register (BJ "carry ... in a CTA loop")          */
    AFFINESCAN_AFFINE_BLELLOCH = 3, /* ABLATION: the paper's shared-memory Blelloch
                                       upsweep / root init / downsweep / reconstruction
                                       (P:103-107), CTA-loop carry             */
    AFFINESCAN_AFFINE_WARP_SEQ = 4, /* one warp per sequence (many short sequences), carry in
                                       a register, no shared memory, no barrier           */
    /* selective_scan_fwd */
    AFFINESCAN_SELECTIVE_WARP_ROW = 11, /* one warp per (b,d) row, lanes own consecutive
                                           chunks of L, warp-shuffle pair scan            */
    AFFINESCAN_SELECTIVE_WARP_ROW_TMA = 13, /* same schedule; a CTA = R rows of one batch
                                               sharing B_t/C_t tiles staged in shared memory
                                               by TMA tensor copies (needs N == 16, 16-byte
                                               aligned pointers, L a multiple of the vector) */
    AFFINESCAN_SELECTIVE_LANE_ROW = 12, /* 1, 2 or 4 lanes per (b,d) row, sequential in L, the
                                           row's states in registers; B/C tiles staged in
                                           shared memory by TMA tensor copies; the grid is
                                           uniform (one or two lanes per row) or balanced
                                           (one CTA per SM, every sub-partition three two-lane
                                           warps and one four-lane warp), chosen from the row
                                           count (needs N == 16, d_inner % 32 == 0, 16-byte
                                           aligned pointers, L a multiple of the vector)   */
    AFFINESCAN_SELECTIVE_CHUNKED = 14   /* few rows x long L: L is cut into chunks that run on
                                           different CTAs; the carry h_in crosses chunks by
                                           decoupled look-back over per-(row, state) chunk
                                           aggregates (BJ "decoupled look-back for very long
                                           sequences"; same shape requirements as WARP_ROW_TMA) */
} affinescan_variant;

/* Structure the caller asserts about A: a hint the
 * library may exploit; the result is what the general kernel computes on the same A. */
typedef enum affinescan_a_structure {
    AFFINESCAN_A_GENERAL = 0,        /* any A[d,n]                                          */
    AFFINESCAN_A_SCALAR_PER_ROW = 1, /* A[d,n] == A[d,0] for every n (one decay per row):
                                        one exp per (b,d,t) instead of N                    */
    AFFINESCAN_A_POWERS = 2          /* A[d,n] == (n+1)*A[d,0] (S4D-real structure):
                                        a_n = r^(n+1), r = exp(delta*A[d,0]): one exp and
                                        N-1 multiplies per (b,d,t)                          */
} affinescan_a_structure;

/* ------------------------------------------------------------------------------------
 * affine_scan — inclusive scan of the affine recurrence
 *
 *     h[s,t] = a[s,t] * h[s,t-1] + u[s,t],   h[s,-1] = h0[s],   t = 0..L-1
 *     h_last[s] = h[s,L-1]                   (= h0[s] when L == 0)
 *
 * i.e. the prefix scan over the pairs (A_t,U_t) = (a_t, b_t x_t) (Eq.6) under
 * (A2,U2)(+)(A1,U1) = (A2 A1, A2 U1 + U2) (Eq.7), which reproduces the
 * sequential recurrence h_t = a_t h_{t-1} + b_t x_t (Eq.1, Eq.3) with the
 * initial state h_0 of P:81 Eq.5.  Also covers the weighted-prefix recurrence
 * h_t = alpha_t h_{t-1} + beta_t (Eq.10) with a = alpha, u = beta.
 *
 *   a, u     [num_seq, L]  io dtype   in
 *   h0       [num_seq]     fp32       in, NULL => 0
 *   h        [num_seq, L]  io dtype   out
 *   h_last   [num_seq]     fp32       out, NULL => not written
 *
 * num_seq == 0 or L == 0 is OK (h_last <- h0 or 0).  Returns an affinescan_status.
 * ------------------------------------------------------------------------------------ */
AFFINESCAN_API int affine_scan(const void* a, const void* u, const float* h0, void* h,
                               float* h_last, int64_t num_seq, int64_t L, int io_dtype,
                               void* cuda_stream);

/* Same, forcing a kernel variant (AFFINESCAN_VARIANT_AUTO or an AFFINESCAN_AFFINE_*). */
AFFINESCAN_API int affine_scan_ex(const void* a, const void* u, const float* h0, void* h,
                                  float* h_last, int64_t num_seq, int64_t L, int io_dtype,
                                  int variant, void* cuda_stream);

/* Same computation with HOST buffers: copies a, u, h0 to the device, runs the kernel,
 * copies h and h_last back, and synchronises `cuda_stream`.  Device staging buffers are
 * owned and cached by the library. */
AFFINESCAN_API int affine_scan_host(const void* a, const void* u, const float* h0, void* h,
                                    float* h_last, int64_t num_seq, int64_t L, int io_dtype,
                                    void* cuda_stream);

/* ------------------------------------------------------------------------------------
 * affine_scan_static_scratch — affine_scan (same arguments, same result as
 * affine_scan_ex(..., AFFINESCAN_AFFINE_LOOKBACK, ...)) for callers that cannot allocate device
 * memory.
 *
 * Why it exists.  The look-back scan needs one 16-byte descriptor per tile for the carry that
 * crosses tiles (prefix compositions under P:90 Eq.7).  affine_scan takes that scratch
 * from cudaMallocAsync.  That is not acceptable everywhere: an inference server that gave all
 * free HBM to its own cache at start-up has nothing left for the driver to hand out; a framework
 * whose allocator must own every byte cannot have a library allocate behind its back; a
 * latency-bound control loop must not meet the driver's allocation lock on its hot path; a
 * plug-in may simply be handed its input and output buffers and forbidden everything else.  This
 * entry point calls no cudaMalloc / cudaMallocAsync / cudaFree and no allocating library
 * routine, ever: the descriptors live in a fixed 1 MiB `static __device__` array inside the
 * library image.  Every GPU on which the library's code is loaded holds that 1 MiB until the
 * process exits, used or not.
 *
 * Limit.  65 535 tiles.  A tile is 4096 elements (fp32) or 8192 elements (bf16) when a, u, h are
 * 16-byte aligned and L is a multiple of 4 (fp32) / 8 (bf16); otherwise the scalar-access
 * kernel runs with 1024-element tiles.  So num_seq*L may be at most 268 431 360 (fp32),
 * 536 862 720 (bf16) or 67 107 840 (scalar fallback):
 * affine_scan_static_scratch_max_elements(io_dtype, vectorised) returns these.  Anything larger
 * returns AFFINESCAN_ERR_TOO_LARGE before any device work; use affine_scan for it.
 *
 * Sharing.  There is ONE array per GPU and every call on that GPU uses it.  It keeps what the
 * previous call wrote; each call zeroes the two counters that must start at zero (an 8-byte
 * cudaMemsetAsync on `cuda_stream`) and relies on the per-launch epoch in the descriptors for the
 * rest.  Calls that can overlap on the GPU — two streams, two host threads, a second process
 * does NOT count (it has its own copy) — RACE on the array and give wrong results or hang:
 * keep all calls on one stream, or order them with events.
 *
 * First call.  The first call on each device looks up the array's device address
 * (cudaGetSymbolAddress, which may make the driver load the library's code onto that device).
 * Make that first call outside any stream capture, with the device current that the later calls
 * will use.
 *
 * Asynchronous on cuda_stream like affine_scan; num_seq == 0 or L == 0 is OK.
 * ------------------------------------------------------------------------------------ */
AFFINESCAN_API int affine_scan_static_scratch(const void* a, const void* u, const float* h0,
                                              void* h, float* h_last, int64_t num_seq, int64_t L,
                                              int io_dtype, void* cuda_stream);
/* Largest num_seq*L affine_scan_static_scratch accepts for io_dtype on its vector path
 * (vectorised != 0) or its scalar-access fallback (vectorised == 0); 0 for an unknown dtype.
 * No device work. */
AFFINESCAN_API int64_t affine_scan_static_scratch_max_elements(int io_dtype, int vectorised);

/* ------------------------------------------------------------------------------------
 * selective_scan_fwd — Mamba-style fused forward selective scan (BJ north_star):
 *
 *     a_t[d,n] = exp(delta_t[d] * A[d,n])              discretisation (BJ)
 *     u_t[d,n] = delta_t[d] * B_t[n] * x_t[d]          b_t = delta_t B_t (BJ); U = b x
 *     h_t[d,n] = a_t[d,n] * h_{t-1}[d,n] + u_t[d,n]    (Eq.3), h_{-1} = h0
 *     y_t[d]   = sum_n C_t[n] * h_t[d,n] + D[d] * x_t[d]   (BJ; Eq.4 is N=1, D=0)
 *
 * h is never written to memory; only y and the final state are.
 *
 *   x, delta [batch, d_inner, L]  io dtype  in   (delta > 0: softplus already applied)
 *   A        [d_inner, N]         fp32      in   (negative => a in (0,1))
 *   B, C     [batch, N, L]        io dtype  in
 *   D        [d_inner]            fp32      in, NULL => no skip term
 *   h0       [batch, d_inner, N]  fp32      in, NULL => 0
 *   y        [batch, d_inner, L]  io dtype  out, NULL => not stored (needs h_last != NULL:
 *                                            the aggregate-only call of the L-sharded scan)
 *   h_last   [batch, d_inner, N]  fp32      out, NULL => not written
 *
 * 1 <= N <= AFFINESCAN_MAX_N (N = 16 is the tuned case).  exp is evaluated as
 * ex2.approx.ftz.f32(delta * (A * log2 e)) (Q11).  batch, d_inner or L == 0 is OK.
 * ------------------------------------------------------------------------------------ */
AFFINESCAN_API int selective_scan_fwd(const void* x, const void* delta, const float* A,
                                      const void* B, const void* C, const float* D,
                                      const float* h0, void* y, float* h_last, int batch,
                                      int d_inner, int N, int64_t L, int io_dtype,
                                      void* cuda_stream);

/* Same, forcing a kernel variant (AUTO or an AFFINESCAN_SELECTIVE_*). */
AFFINESCAN_API int selective_scan_fwd_ex(const void* x, const void* delta, const float* A,
                                         const void* B, const void* C, const float* D,
                                         const float* h0, void* y, float* h_last, int batch,
                                         int d_inner, int N, int64_t L, int io_dtype,
                                         int variant, void* cuda_stream);

/* Same computation with HOST buffers (see affine_scan_host).  Pipelined over batches: the H2D
 * copy of batch b+1, the kernel of batch b and the D2H copy of batch b-1 overlap on internal
 * copy streams (pinned host memory is needed for the overlap; pageable memory still works). */
AFFINESCAN_API int selective_scan_fwd_host(const void* x, const void* delta, const float* A,
                                           const void* B, const void* C, const float* D,
                                           const float* h0, void* y, float* h_last,
                                           int batch, int d_inner, int N, int64_t L,
                                           int io_dtype, void* cuda_stream);

/* ------------------------------------------------------------------------------------
 * selective_scan_fwd_ext — selective_scan_fwd with the steps either side of the scan that a
 * production selective-scan kernel fuses beyond the affine recurrence ("integrates
 * recurrence, projection, and gating") and the reset mechanism the paper leaves
 * unmodelled.  Every extra pointer may be NULL (=> that step is absent); with all of
 * them NULL and delta_softplus == 0 this is selective_scan_fwd_ex.
 *
 *     Delta_t[d] = softplus(delta_t[d] + delta_bias[d])    if delta_softplus != 0
 *                = delta_t[d] + delta_bias[d]              otherwise
 *     reset[b,t] != 0  =>  step t starts a new sequence: h_{t-1} := 0, i.e. the transition
 *                          pair of step t is (0, u_t), a left zero of (+) (Eq.7); with
 *                          reset[b,0] != 0 the initial state h0 of that batch is ignored.
 *                          Packs several variable-length sequences along L.
 *     a_t, u_t, h_t, y_t as in selective_scan_fwd with Delta_t
 *     y_t[d] <- y_t[d] * silu(z_t[d]),   silu(v) = v / (1 + exp(-v))          if z != NULL
 *
 *   z           [batch, d_inner, L]  io dtype   in, NULL => no gate
 *   delta_bias  [d_inner]            fp32       in, NULL => 0
 *   reset       [batch, L]           uint8      in, NULL => no resets
 *   a_structure an affinescan_a_structure the caller asserts about A (0 = general)
 *   variant     AFFINESCAN_VARIANT_AUTO or an AFFINESCAN_SELECTIVE_*
 * softplus(v) is evaluated as max(v, 0) + log1p(e) with e = 2^(-|v| log2 e) in (0, 1] (MUFU.EX2):
 * log1p(e) = log2(1 + e) ln 2 (MUFU.LG2) for e >= 0.01 and the series e - e^2/2 + e^3/3 below
 * that, so it is finite for every v and a tiny Delta keeps its relative accuracy; silu with
 * MUFU.EX2 / MUFU.RCP (fp32 io) or one MUFU.TANH (bf16 io).
 * ------------------------------------------------------------------------------------ */
AFFINESCAN_API int selective_scan_fwd_ext(const void* x, const void* delta, const float* A,
                                          const void* B, const void* C, const float* D,
                                          const void* z, const float* delta_bias,
                                          const uint8_t* reset, const float* h0, void* y,
                                          float* h_last, int batch, int d_inner, int N,
                                          int64_t L, int io_dtype, int delta_softplus,
                                          int a_structure, int variant, void* cuda_stream);

/* Same computation with HOST buffers (see selective_scan_fwd_host). */
AFFINESCAN_API int selective_scan_fwd_ext_host(const void* x, const void* delta, const float* A,
                                               const void* B, const void* C, const float* D,
                                               const void* z, const float* delta_bias,
                                               const uint8_t* reset, const float* h0, void* y,
                                               float* h_last, int batch, int d_inner, int N,
                                               int64_t L, int io_dtype, int delta_softplus,
                                               int a_structure, void* cuda_stream);

/* The gated form of a Mamba block: Delta = softplus(delta_raw + delta_bias[d])
 * as a prologue and y <- y * silu(z) as an epilogue of the same kernel (no extra pass over
 * HBM).  delta_bias and z may be NULL.  Equals selective_scan_fwd_ext(..., reset = NULL,
 * delta_softplus = 1, AFFINESCAN_A_GENERAL, AFFINESCAN_VARIANT_AUTO). */
AFFINESCAN_API int selective_scan_fwd_gated(const void* x, const void* delta_raw,
                                            const float* delta_bias, const float* A,
                                            const void* B, const void* C, const float* D,
                                            const void* z, const float* h0, void* y,
                                            float* h_last, int batch, int d_inner, int N,
                                            int64_t L, int io_dtype, void* cuda_stream);

/* reset[t] = 1 where a packed sequence starts (t = cu_seqlens[i], i = 0..num_seq-1; entries
 * outside [0, L) are ignored), 0 elsewhere.  cu_seqlens: [num_seq] int32, device; reset: [L]
 * uint8, device (one batch row of selective_scan_fwd_ext's reset).  Asynchronous on the stream. */
AFFINESCAN_API int affinescan_reset_mask_from_cu_seqlens(const int32_t* cu_seqlens, int num_seq,
                                                         uint8_t* reset, int64_t L,
                                                         void* cuda_stream);

/* ------------------------------------------------------------------------------------
 * L-sharded scan across GPUs (the paper "does not yet address distributed or
 * multi-GPU scan execution").  Rank r of R holds the L-slice [t_r, t_{r+1}) of every
 * tensor.  The path has ONE exchange step:
 *   1. selective_scan_slice_aggregate: the slice's transition pair per (row, state),
 *        P = prod_t a_t = exp(A * sum_t delta_t),  U = state after the slice when entered with 0
 *      (the total composition of the slice's pairs);
 *   2. all-gather of (P, U) over the ranks (rows*N*2 floats per rank: NCCL, by the caller);
 *   3. affinescan_compose_carry: h_in = (P_{r-1},U_{r-1}) (+) ... (+) (P_0,U_0) applied to h0
 *      (Eq.7);
 *   4. selective_scan_fwd on the slice with h0 = h_in (rank 0 can skip 1-3 and use h0).
 * paper_2606_00601_b200/sharding.py drives the four steps over torch.distributed (rank 0 skips
 * 3, the last rank skips 1).  `delta` here is the step size that enters the recurrence: the
 * softplus/bias prologue, gate and resets of selective_scan_fwd_ext are NOT part of the slice
 * aggregate, so apply them before sharding or do not shard the extended forward.
 *
 *   P, U      [batch, d_inner, N] fp32  out          (selective_scan_slice_aggregate)
 *   P_all, U_all [world, n] fp32 in; h0 [n] fp32 in or NULL; h_in [n] fp32 out; n = rows*N
 * ------------------------------------------------------------------------------------ */
AFFINESCAN_API int selective_scan_slice_aggregate(const void* x, const void* delta, const float* A,
                                                  const void* B, const void* C, float* P, float* U,
                                                  int batch, int d_inner, int N, int64_t L,
                                                  int io_dtype, void* cuda_stream);
AFFINESCAN_API int affinescan_compose_carry(const float* P_all, const float* U_all,
                                            const float* h0, float* h_in, int rank, int world,
                                            int64_t n, void* cuda_stream);

/* ------------------------------------------------------------------------------------
 * selective_scan_bwd — backward pass of selective_scan_fwd (the paper evaluates
 * "forward selective-scan workloads" only).  For the scalar
 *     loss = sum dy[b,d,t] y[b,d,t] + sum dh_last[b,d,n] h_last[b,d,n]
 * it writes d loss / d(input) for every input of selective_scan_fwd.  The adjoint of
 * h_t = a_t h_{t-1} + u_t (Eq.3) is the same affine recurrence run right to left,
 * g_t = a_{t+1} g_{t+1} + C_t dy_t, i.e. the scan of P:90 Eq.(7) over the reversed sequence;
 * h_{t-1} is recomputed from checkpoints kept in library scratch (8 B per (b,d,t) for the
 * checkpoints + 8 B for the dB/dC partial sums, stream-ordered), never divided out.
 *
 *   x, delta, dy [batch, d_inner, L] io dtype  in      A [d_inner, N] fp32   in
 *   B, C         [batch, N, L]       io dtype  in      D [d_inner]    fp32   in, NULL => 0
 *   h0, dh_last  [batch, d_inner, N] fp32      in, NULL => 0
 *   dx, ddelta   [batch, d_inner, L] fp32      out     dA [d_inner, N] fp32  out (sum over batch)
 *   dB, dC       [batch, N, L]       fp32      out (sum over d_inner)
 *   dD           [d_inner]           fp32      out (sum over batch)
 *   dh0          [batch, d_inner, N] fp32      out
 * Every output pointer may be NULL (=> not written).  All gradients are fp32 whatever the io
 * dtype; sums over rows and batches are formed in a fixed order (bitwise reproducible).
 * Supported shapes: N == 16, d_inner % 32 == 0, L % 8 == 0, batch <= 65535, 16-byte aligned
 * pointers (dx and ddelta included); anything else returns AFFINESCAN_ERR_UNSUPPORTED before any
 * device work.  This is the backward of the PLAIN forward only: selective_scan_fwd_ext /
 * _gated (softplus/bias prologue, silu(z) gate, resets) have no backward here — differentiate
 * those steps outside (dz, dbias and the softplus factor on ddelta are elementwise).
 * Asynchronous on cuda_stream.
 * ------------------------------------------------------------------------------------ */
AFFINESCAN_API int selective_scan_bwd(const void* x, const void* delta, const float* A,
                                      const void* B, const void* C, const float* D,
                                      const float* h0, const void* dy, const float* dh_last,
                                      float* dx, float* ddelta, float* dA, float* dB, float* dC,
                                      float* dD, float* dh0, int batch, int d_inner, int N,
                                      int64_t L, int io_dtype, void* cuda_stream);

/* Same with a CALLER-PROVIDED workspace, so that the caller's own allocator owns (and can cache,
 * account for and reclaim) the ~16 bytes per (b,d,t) the backward pass needs: `workspace` is a
 * device buffer of at least selective_scan_bwd_workspace_bytes(batch, d_inner, N, L) bytes,
 * 16-byte aligned, used from the call until its kernels finish on cuda_stream; contents on
 * entry do not matter and are garbage afterwards.  workspace == NULL => selective_scan_bwd
 * (per-call cudaMallocAsync).  A buffer that is too small or misaligned returns
 * AFFINESCAN_ERR_TOO_LARGE before any device work.  With a workspace the call allocates
 * nothing. */
AFFINESCAN_API int selective_scan_bwd_ws(const void* x, const void* delta, const float* A,
                                         const void* B, const void* C, const float* D,
                                         const float* h0, const void* dy, const float* dh_last,
                                         float* dx, float* ddelta, float* dA, float* dB, float* dC,
                                         float* dD, float* dh0, int batch, int d_inner, int N,
                                         int64_t L, int io_dtype, void* workspace,
                                         int64_t workspace_bytes, void* cuda_stream);
/* Bytes of workspace selective_scan_bwd needs for this shape; 0 for an empty or unsupported
 * shape.  No device work. */
AFFINESCAN_API int64_t selective_scan_bwd_workspace_bytes(int batch, int d_inner, int N, int64_t L);

/* ------------------------------------------------------------------------------------
 * Introspection (no device work)
 * ------------------------------------------------------------------------------------ */
/* Static, NUL-terminated description of a status code. */
AFFINESCAN_API const char* affinescan_status_string(int status);
/* cudaError_t of the last AFFINESCAN_ERR_CUDA on the calling thread (0 if none). */
AFFINESCAN_API int affinescan_last_cuda_error(void);
/* affinescan_variant the last successful call on the calling thread ran (0 if none or
 * if the call was a no-op on an empty shape). */
AFFINESCAN_API int affinescan_last_variant(void);
/* Number of kernel launches this process has issued through the library so far. */
AFFINESCAN_API int64_t affinescan_launch_count(void);
/* Number of look-back scratch buffers the library currently caches on the current device
 * (never more than 64; see the conventions at the top). */
AFFINESCAN_API int affinescan_cached_scratch_buffers(void);
/* Library version: major*10000 + minor*100 + patch. */
AFFINESCAN_API int affinescan_version(void);
/* Tuning knobs for ablations and sweeps (process-wide; -1 restores the default chosen from
 * the shape).  Returns AFFINESCAN_ERR_UNSUPPORTED for an unknown key or value. */
typedef enum affinescan_option {
    AFFINESCAN_OPT_LANE_ROW_G = 1,      /* lane_row grid: 1 or 2 lanes per (b,d) row; 3 = balanced mix */
    AFFINESCAN_OPT_LANE_ROW_POLY16 = 2, /* sixteenths (0 or 4) of the exponentials evaluated by
                                           the fma-pipe polynomial instead of MUFU.EX2 (one-lane
                                           grid only; the other grids ignore it)                 */
    AFFINESCAN_OPT_DETERMINISTIC = 3    /* 1: AFFINESCAN_VARIANT_AUTO never picks a decoupled
                                           look-back schedule (AFFINE_LOOKBACK, SELECTIVE_CHUNKED),
                                           so every default call is bitwise reproducible run to
                                           run, at the price of speed on few long sequences / few
                                           rows; 0 or -1 (default): fastest schedule.  A forced
                                           variant is never overridden.                          */
} affinescan_option;
AFFINESCAN_API int affinescan_set_option(int key, int value);
/* Frees the cached scratch / staging buffers, copy streams and events of the current device
 * (synchronises it).  Must not run concurrently with other calls into the library. */
AFFINESCAN_API int affinescan_release_cache(void);

#ifdef __cplusplus
}
#endif
#endif /* AFFINESCAN_H_ */
