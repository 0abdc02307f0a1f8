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
