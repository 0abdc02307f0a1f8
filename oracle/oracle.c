/*
 * oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, sequential float64 CPU statement of what libaffinescan computes,
 * written from /root/reference/PAPER.md (arxiv/paper_2606_00601, "ScanWeaver";
 * cited below as P:<line>) and from BASELINE.json's north_star (cited as BJ)
 * where the paper is silent.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this file.  It shares
 * no code, header, table or helper with paper_2606_00601_b200/ (the CUDA path).
 *
 * Every function takes HOST pointers to dense row-major float64 arrays (the
 * callers widen fp32 / bf16 storage to float64 exactly, so input rounding is
 * never counted as error) and returns nothing; sizes are int64.
 *
 * Parity pins (tests/test_oracle_pins.py, run with -m "not gpu"):
 *   oracle_affine_scan        : a==1 prefix sum, u==0 running product, geometric
 *                               series, Eq.5 in exact rational arithmetic, split
 *                               invariance, linearity               -> pinned
 *   oracle_compose / fold     : every bracketing of <=8 pairs (Catalan trees) in
 *                               exact dyadic arithmetic; h_last identity -> pinned
 *   oracle_selective_scan_fwd : N=1,C=1 reduction to the affine scan, delta==0,
 *                               A->0 cumulative sum, independent closed-form
 *                               (cumsum/exp-of-differences) evaluation -> pinned
 *   oracle_blelloch_scan      : equals the sequential loop bit-for-bit on dyadic
 *                               inputs, power-of-two and padded sizes  -> pinned
 *   oracle_selective_scan_fwd_ext : bitwise equal to oracle_selective_scan_fwd with
 *                               every option off; softplus / silu against math-library
 *                               closed forms; bias -> -inf holds the state; a reset
 *                               at t equals two independent calls split at t -> pinned
 *   oracle_selective_scan_bwd : central finite differences of the (pinned) forward
 *                               oracle in every input; adjoint identity
 *                               <dy, J v> = <J^T dy, v>                  -> pinned
 * Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------- *
 * Sequential affine recurrence, Eq.(1), Eq.(2), Eq.(3):
 *     h_t = a_t * h_{t-1} + u_t ,   u_t = b_t * x_t  (Eq.(6), U_t = b_t x_t)
 * with the initial state h_0 of P:81 Eq.(5).  Arrays are 0-based: h[s][t] is the
 * paper's h_{t+1}; the result is the INCLUSIVE scan (reading Q1).
 *     a, u : [S][L]      h0 : [S] or NULL (=> 0)
 *     h    : [S][L]      h_last : [S] or NULL ; h_last[s] = h[s][L-1] (h0 if L==0)
 * ------------------------------------------------------------------------- */
void oracle_affine_scan(const double *a, const double *u, const double *h0,
                        double *h, double *h_last, int64_t S, int64_t L)
{
    for (int64_t s = 0; s < S; ++s) {
        double hp = h0 ? h0[s] : 0.0;
        for (int64_t t = 0; t < L; ++t) {
            hp = a[s * L + t] * hp + u[s * L + t];
            h[s * L + t] = hp;
        }
        if (h_last) h_last[s] = hp;
    }
}

/* ------------------------------------------------------------------------- *
 * Mamba-style selective-scan forward (BJ north_star; the paper's Eq.(3)-(4),
 * P:69-73, with the discretisation and output BJ fixes — DESIGN.md Q5/Q6):
 *     a_t[d,n] = exp(delta_t[d] * A[d,n])          (BJ: a_t = exp(Δ_t·A))
 *     u_t[d,n] = (delta_t[d] * B_t[n]) * x_t[d]    (BJ: b_t = Δ_t·B_t ; P:86 U=b x)
 *     h_t[d,n] = a_t[d,n] * h_{t-1}[d,n] + u_t[d,n]            (Eq.(3))
 *     y_t[d]   = sum_n C_t[n] * h_t[d,n] + D[d] * x_t[d]       (BJ; P:73 is N=1,D=0)
 * Layouts (Q8): x, delta, y [batch][d_inner][L]; A [d_inner][N];
 * B, C [batch][N][L]; D [d_inner] or NULL; h0, h_last [batch][d_inner][N] or NULL.
 * exp is libm's double exp.  The n-sum runs n = 0..N-1 in order.
 * ------------------------------------------------------------------------- */
void oracle_selective_scan_fwd(const double *x, const double *delta, const double *A,
                               const double *B, const double *C, const double *D,
                               const double *h0, double *y, double *h_last,
                               int64_t batch, int64_t d_inner, int64_t N, int64_t L)
{
    double *hs = (double *)malloc((size_t)(N > 0 ? N : 1) * sizeof(double));
    for (int64_t b = 0; b < batch; ++b) {
        for (int64_t d = 0; d < d_inner; ++d) {
            const int64_t row = b * d_inner + d;
            for (int64_t n = 0; n < N; ++n) hs[n] = h0 ? h0[row * N + n] : 0.0;
            for (int64_t t = 0; t < L; ++t) {
                const double dl = delta[row * L + t];
                const double xv = x[row * L + t];
                double acc = 0.0;
                for (int64_t n = 0; n < N; ++n) {
                    const double at = exp(dl * A[d * N + n]);
                    const double ut = (dl * B[(b * N + n) * L + t]) * xv;
                    hs[n] = at * hs[n] + ut;
                    acc += C[(b * N + n) * L + t] * hs[n];
                }
                y[row * L + t] = acc + (D ? D[d] * xv : 0.0);
            }
            if (h_last)
                for (int64_t n = 0; n < N; ++n) h_last[row * N + n] = hs[n];
        }
    }
    free(hs);
}

/* ------------------------------------------------------------------------- *
 * Associative composition of affine pairs, Eq.(7):
 *     (A2,U2) (+) (A1,U1) = (A2*A1, A2*U1 + U2)
 * The LEFT operand is the LATER transition (Q2); not commutative.
 * ------------------------------------------------------------------------- */
void oracle_compose(double A2, double U2, double A1, double U1,
                    double *A_out, double *U_out)
{
    *A_out = A2 * A1;
    *U_out = A2 * U1 + U2;
}

/* Left fold e_{L-1} (+) ( ... (+) (e_1 (+) e_0)) of the pairs e_t = (a_t, u_t)
 * ("each prefix composition produces the affine transformation
 * corresponding to a recurrence segment").  L == 0 gives the identity (1, 0). */
void oracle_fold_pairs(const double *a, const double *u, int64_t L,
                       double *A_tot, double *U_tot)
{
    double At = 1.0, Ut = 0.0;
    for (int64_t t = 0; t < L; ++t) oracle_compose(a[t], u[t], At, Ut, &At, &Ut);
    *A_tot = At;
    *U_tot = Ut;
}

/* ------------------------------------------------------------------------- *
 * CPU model of the paper's Blelloch schedule for ONE
 * sequence, used to check the shared-memory ablation kernel's structure:
 *   upsweep (tree reduction)  ->  root initialisation  ->  downsweep (prefix
 *   propagation)  ->  affine-prefix reconstruction.
 * The paper names the phases but not their details for a non-commutative
 * operator; Q3/Q4/Q16 fix them: identity (1,0) at the root and as
 * padding up to the next power of two; upsweep  x[r] <- x[r] (+) x[l]  (r later);
 * downsweep  t <- x[l]; x[l] <- x[r]; x[r] <- t (+) x[r]_old ; reconstruction
 * incl_t = e_t (+) excl_t and h_t = A_incl * h0 + U_incl.
 *     a, u : [L]   h0 : scalar   h : [L]
 * ------------------------------------------------------------------------- */
void oracle_blelloch_scan(const double *a, const double *u, double h0, double *h,
                          int64_t L)
{
    if (L <= 0) return;
    int64_t P2 = 1;
    while (P2 < L) P2 <<= 1;
    double *TA = (double *)malloc((size_t)P2 * sizeof(double));
    double *TU = (double *)malloc((size_t)P2 * sizeof(double));
    for (int64_t i = 0; i < P2; ++i) {
        TA[i] = i < L ? a[i] : 1.0; /* identity padding (Q3) */
        TU[i] = i < L ? u[i] : 0.0;
    }
    /* upsweep */
    for (int64_t stride = 1; stride < P2; stride <<= 1) {
        for (int64_t r = 2 * stride - 1; r < P2; r += 2 * stride) {
            const int64_t l = r - stride;
            oracle_compose(TA[r], TU[r], TA[l], TU[l], &TA[r], &TU[r]);
        }
    }
    /* root initialisation */
    TA[P2 - 1] = 1.0;
    TU[P2 - 1] = 0.0;
    /* downsweep */
    for (int64_t stride = P2 >> 1; stride >= 1; stride >>= 1) {
        for (int64_t r = 2 * stride - 1; r < P2; r += 2 * stride) {
            const int64_t l = r - stride;
            const double lA = TA[l], lU = TU[l];
            TA[l] = TA[r];
            TU[l] = TU[r];
            oracle_compose(lA, lU, TA[r], TU[r], &TA[r], &TU[r]);
        }
    }
    /* affine-prefix reconstruction: TA/TU now hold the EXCLUSIVE prefixes */
    for (int64_t t = 0; t < L; ++t) {
        double Ai, Ui;
        oracle_compose(a[t], u[t], TA[t], TU[t], &Ai, &Ui);
        h[t] = Ai * h0 + Ui;
    }
    free(TA);
    free(TU);
}

/* ------------------------------------------------------------------------- *
 * Extended forward: the steps either side of the scan that
 * the paper names as what a production selective-scan kernel fuses beyond the
 * affine recurrence ("integrates recurrence, projection, and gating";
 * P:290 "additional fused operations beyond the affine recurrence") and the
 * reset mechanism it leaves unmodelled:
 *     Delta_t[d] = softplus(delta_t[d] + delta_bias[d])     if delta_softplus
 *                = delta_t[d] + delta_bias[d]               otherwise
 *     reset[b,t] != 0  =>  step t starts a new sequence: h_{t-1} := 0, i.e. the
 *                          transition pair of step t is (0, u_t), a left zero of
 *                          (+) (Eq.(7))
 *     a_t, u_t, h_t, y_t as in oracle_selective_scan_fwd with Delta_t
 *     y_t[d] <- y_t[d] * silu(z_t[d]),  silu(v) = v / (1 + exp(-v))      if z
 * softplus(v) = log(1 + exp(v)), written max(v,0) + log1p(exp(-|v|)) (the same
 * function, finite for every v).
 *   delta_bias : [d_inner] or NULL (=> 0)      z : [batch][d_inner][L] or NULL
 *   reset      : [batch][L] or NULL, nonzero = start of a sequence
 * ------------------------------------------------------------------------- */
static double oracle_softplus(double v)
{
    return (v > 0.0 ? v : 0.0) + log1p(exp(-fabs(v)));
}

void oracle_selective_scan_fwd_ext(const double *x, const double *delta, const double *A,
                                   const double *B, const double *C, const double *D,
                                   const double *z, const double *delta_bias,
                                   const double *reset, const double *h0, double *y,
                                   double *h_last, int64_t batch, int64_t d_inner, int64_t N,
                                   int64_t L, int64_t delta_softplus)
{
    double *hs = (double *)malloc((size_t)(N > 0 ? N : 1) * sizeof(double));
    for (int64_t b = 0; b < batch; ++b) {
        for (int64_t d = 0; d < d_inner; ++d) {
            const int64_t row = b * d_inner + d;
            for (int64_t n = 0; n < N; ++n) hs[n] = h0 ? h0[row * N + n] : 0.0;
            for (int64_t t = 0; t < L; ++t) {
                double dl = delta[row * L + t] + (delta_bias ? delta_bias[d] : 0.0);
                if (delta_softplus) dl = oracle_softplus(dl);
                const double xv = x[row * L + t];
                if (reset && reset[b * L + t] != 0.0)
                    for (int64_t n = 0; n < N; ++n) hs[n] = 0.0;
                double acc = 0.0;
                for (int64_t n = 0; n < N; ++n) {
                    const double at = exp(dl * A[d * N + n]);
                    const double ut = (dl * B[(b * N + n) * L + t]) * xv;
                    hs[n] = at * hs[n] + ut;
                    acc += C[(b * N + n) * L + t] * hs[n];
                }
                double yv = acc + (D ? D[d] * xv : 0.0);
                if (z) {
                    const double zv = z[row * L + t];
                    yv *= zv / (1.0 + exp(-zv));
                }
                y[row * L + t] = yv;
            }
            if (h_last)
                for (int64_t n = 0; n < N; ++n) h_last[row * N + n] = hs[n];
        }
    }
    free(hs);
}

/* ------------------------------------------------------------------------- *
 * Backward pass of oracle_selective_scan_fwd (the paper evaluates
 * "forward selective-scan workloads" only).  For the scalar
 *     loss = sum dy[b,d,t]*y[b,d,t] + sum dh_last[b,d,n]*h_last[b,d,n]
 * it returns d loss / d(input) for every input.  The adjoint of the recurrence
 * h_t = a_t h_{t-1} + u_t (Eq.(3)) is the same affine recurrence run from
 * right to left,
 *     g_t = a_{t+1} g_{t+1} + C_t dy_t ,   g_{L-1} = dh_last + C_{L-1} dy_{L-1},
 * with g_t = d loss / d h_t; then, with a_t = exp(Delta_t A), u_t = Delta_t B_t x_t:
 *     dC_t[n]    += dy_t h_t[n]                        (summed over d)
 *     dD[d]      += dy_t x_t
 *     dx_t        = D dy_t + sum_n g_t[n] Delta_t B_t[n]
 *     dB_t[n]    += g_t[n] Delta_t x_t                 (summed over d)
 *     dDelta_t    = sum_n g_t[n] (A[n] a_t[n] h_{t-1}[n] + B_t[n] x_t)
 *     dA[d,n]    += g_t[n] Delta_t a_t[n] h_{t-1}[n]
 *     dh0[n]      = a_0[n] g_0[n]
 * One row at a time: a forward sweep that keeps every h_t of the row, then the
 * reverse sweep.  Outputs may be NULL (skipped); dA, dB, dC, dD are ZEROED here.
 *   dy [batch][d_inner][L]; dh_last [batch][d_inner][N] or NULL (=> 0)
 *   dx, ddelta [batch][d_inner][L]; dA [d_inner][N]; dB, dC [batch][N][L];
 *   dD [d_inner]; dh0 [batch][d_inner][N]
 * ------------------------------------------------------------------------- */
void oracle_selective_scan_bwd(const double *x, const double *delta, const double *A,
                               const double *B, const double *C, const double *D,
                               const double *h0, const double *dy, const double *dh_last,
                               double *dx, double *ddelta, double *dA, double *dB, double *dC,
                               double *dD, double *dh0, int64_t batch, int64_t d_inner,
                               int64_t N, int64_t L)
{
    if (dA) memset(dA, 0, (size_t)(d_inner * N) * sizeof(double));
    if (dB) memset(dB, 0, (size_t)(batch * N * L) * sizeof(double));
    if (dC) memset(dC, 0, (size_t)(batch * N * L) * sizeof(double));
    if (dD) memset(dD, 0, (size_t)d_inner * sizeof(double));
    /* H[t+1][n] = h_t[n]; H[0][n] = h_{-1}[n] = h0 */
    double *H = (double *)malloc((size_t)((L + 1) * (N > 0 ? N : 1)) * sizeof(double));
    double *g = (double *)malloc((size_t)(N > 0 ? N : 1) * sizeof(double));
    for (int64_t b = 0; b < batch; ++b) {
        for (int64_t d = 0; d < d_inner; ++d) {
            const int64_t row = b * d_inner + d;
            for (int64_t n = 0; n < N; ++n) H[n] = h0 ? h0[row * N + n] : 0.0;
            for (int64_t t = 0; t < L; ++t) {
                const double dl = delta[row * L + t];
                const double xv = x[row * L + t];
                for (int64_t n = 0; n < N; ++n) {
                    const double at = exp(dl * A[d * N + n]);
                    const double ut = (dl * B[(b * N + n) * L + t]) * xv;
                    H[(t + 1) * N + n] = at * H[t * N + n] + ut;
                }
            }
            for (int64_t n = 0; n < N; ++n) g[n] = dh_last ? dh_last[row * N + n] : 0.0;
            for (int64_t t = L - 1; t >= 0; --t) {
                const double dl = delta[row * L + t];
                const double xv = x[row * L + t];
                const double dyv = dy[row * L + t];
                double dxv = D ? D[d] * dyv : 0.0;
                double ddl = 0.0;
                if (dD) dD[d] += dyv * xv;
                for (int64_t n = 0; n < N; ++n) {
                    const int64_t bn = (b * N + n) * L + t;
                    const double at = exp(dl * A[d * N + n]);
                    const double hprev = H[t * N + n];
                    /* g[n] holds a_{t+1} g_{t+1}; add this step's direct term */
                    g[n] += C[bn] * dyv;
                    if (dC) dC[bn] += dyv * H[(t + 1) * N + n];
                    dxv += g[n] * dl * B[bn];
                    if (dB) dB[bn] += g[n] * dl * xv;
                    ddl += g[n] * (A[d * N + n] * at * hprev + B[bn] * xv);
                    if (dA) dA[d * N + n] += g[n] * dl * at * hprev;
                    g[n] = at * g[n];   /* carried to step t-1 (and to h0 at t = 0) */
                }
                if (dx) dx[row * L + t] = dxv;
                if (ddelta) ddelta[row * L + t] = ddl;
            }
            if (dh0)
                for (int64_t n = 0; n < N; ++n) dh0[row * N + n] = g[n];
        }
    }
    free(H);
    free(g);
}
