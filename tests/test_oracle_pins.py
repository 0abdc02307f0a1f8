"""Pins for the CPU oracle (oracle/oracle.c) against things that are NOT the oracle:
closed forms, exact rational arithmetic, brute-force bracketings and independent
closed-form evaluations.  CPU only.  Citations: P:<line> = /root/reference/PAPER.md,
BJ = BASELINE.json north_star.  A plausible slip anywhere in the oracle (dropped
term, wrong sign/index, transposed operand, exclusive-vs-inclusive) fails one of
these.
"""
import itertools
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle

RNG = np.random.default_rng(20260602)


# ----------------------------------------------------------------- helpers (exact)
def dyadic(rng, shape, denom=8, lo=-8, hi=8):
    """Small dyadic rationals k/denom: sums/products of a few of them are exact in fp64."""
    return rng.integers(lo, hi + 1, size=shape).astype(np.float64) / denom


def eq5_exact(a, u, h0):
    """P:81 Eq.(5) evaluated literally, O(L²), in exact rational arithmetic.
    h_t = (prod_{i=1..t} a_i) h_0 + sum_{k=1..t} (prod_{i=k+1..t} a_i) b_k x_k, with 1-based
    paper indices mapped to 0-based arrays (a_i -> a[i-1]); returns h_1..h_L."""
    L = len(a)
    fa = [Fraction(float(v)) for v in a]
    fu = [Fraction(float(v)) for v in u]
    out = []
    for t in range(1, L + 1):
        acc = Fraction(float(h0))
        for i in range(1, t + 1):
            acc *= fa[i - 1]
        for k in range(1, t + 1):
            term = fu[k - 1]
            for i in range(k + 1, t + 1):
                term *= fa[i - 1]
            acc += term
        out.append(acc)
    return out


def all_bracketings(pairs):
    """Every binary tree over the ordered list pairs[0..m-1] (index 0 = EARLIEST), combined
    with Eq.(7) written out here in exact Fractions — not via the oracle.  Yields (A, U)."""
    if len(pairs) == 1:
        yield pairs[0]
        return
    for split in range(1, len(pairs)):
        for (A1, U1) in all_bracketings(pairs[:split]):       # earlier segment
            for (A2, U2) in all_bracketings(pairs[split:]):   # later segment
                yield (A2 * A1, A2 * U1 + U2)                 # P:90 Eq.(7)


# ------------------------------------------------------------ affine scan: closed forms
def test_a_equal_one_is_prefix_sum():
    """BJ: a≡1 gives a prefix sum (integer-valued u: exact)."""
    S, L = 3, 257
    u = RNG.integers(-50, 50, size=(S, L)).astype(np.float64)
    h0 = np.array([0.0, 7.0, -3.0])
    h, h_last = oracle.affine_scan(np.ones((S, L)), u, h0)
    assert np.array_equal(h, h0[:, None] + np.cumsum(u, axis=1))
    assert np.array_equal(h_last, h[:, -1])


def test_u_equal_zero_is_running_product():
    """BJ: u≡0 gives a running product; a=0.5 makes every value an exact power of two."""
    L = 60
    h, h_last = oracle.affine_scan(np.full((1, L), 0.5), np.zeros((1, L)), np.array([3.0]))
    assert np.array_equal(h[0], 3.0 * 0.5 ** np.arange(1, L + 1))
    assert h_last[0] == 3.0 * 0.5 ** L
    a = RNG.uniform(0.5, 0.99, size=(2, 100))
    h, _ = oracle.affine_scan(a, np.zeros_like(a), np.array([1.0, -2.0]))
    np.testing.assert_allclose(h, np.array([[1.0], [-2.0]]) * np.cumprod(a, axis=1), rtol=1e-13)


def test_constant_a_is_geometric_series():
    """BJ: constant a,u gives h_t = a^{t+1} h0 + u (1-a^{t+1})/(1-a) (0-based t)."""
    L = 500
    for a0, u0, h00 in [(0.9, 1.5, 0.0), (0.5, -2.0, 4.0), (0.999, 0.01, -1.0)]:
        h, _ = oracle.affine_scan(np.full((1, L), a0), np.full((1, L), u0), np.array([h00]))
        t1 = np.arange(1, L + 1)
        ref = a0 ** t1 * h00 + u0 * (1.0 - a0 ** t1) / (1.0 - a0)
        np.testing.assert_allclose(h[0], ref, rtol=1e-11, atol=1e-13)


def test_eq5_exact_rational():
    """P:81 Eq.(5), literal double loop in Fractions, equals the oracle bit for bit on dyadic
    inputs (every intermediate is exactly representable for L ≤ 12, denominators ≤ 2^39)."""
    for L in (1, 2, 3, 7, 12):
        a = dyadic(RNG, L, denom=8, lo=-7, hi=7)
        u = dyadic(RNG, L, denom=8)
        h0 = 1.25
        h, h_last = oracle.affine_scan(a[None], u[None], np.array([h0]))
        ref = eq5_exact(a, u, h0)
        assert [Fraction(v) for v in h[0]] == ref
        assert Fraction(h_last[0]) == ref[-1]


def test_eq5_random_floats_close():
    """Eq.(5) in Fractions on non-dyadic inputs: the loop is within fp64 rounding."""
    L = 40
    a = RNG.uniform(0.5, 0.99, size=L)
    u = RNG.normal(size=L)
    h, _ = oracle.affine_scan(a[None], u[None], np.array([0.3]))
    ref = np.array([float(v) for v in eq5_exact(a, u, 0.3)])
    np.testing.assert_allclose(h[0], ref, rtol=1e-13, atol=1e-15)


def test_inclusive_not_exclusive_and_index_base():
    """Reading Q1: h[t] includes u[t]; h[0] = a[0]*h0 + u[0]."""
    a = np.array([[2.0, 3.0, 5.0]])
    u = np.array([[1.0, 10.0, 100.0]])
    h, h_last = oracle.affine_scan(a, u, np.array([7.0]))
    assert h[0].tolist() == [15.0, 55.0, 375.0]
    assert h_last[0] == 375.0
    h, _ = oracle.affine_scan(a, u, None)            # h0 = NULL => 0
    assert h[0].tolist() == [1.0, 13.0, 165.0]


def test_empty_length():
    h, h_last = oracle.affine_scan(np.zeros((2, 0)), np.zeros((2, 0)), np.array([4.0, 5.0]))
    assert h.shape == (2, 0) and h_last.tolist() == [4.0, 5.0]


def test_sequences_are_independent():
    a = RNG.uniform(0.5, 0.99, size=(4, 33))
    u = RNG.normal(size=(4, 33))
    h0 = RNG.normal(size=4)
    h, hl = oracle.affine_scan(a, u, h0)
    for s in range(4):
        hs, hls = oracle.affine_scan(a[s:s + 1], u[s:s + 1], h0[s:s + 1])
        assert np.array_equal(hs[0], h[s]) and hls[0] == hl[s]


# ----------------------------------------------------- composition ⊕ and associativity
def test_compose_matches_eq7_and_is_not_commutative():
    """P:90 Eq.(7): (A2,U2)⊕(A1,U1) = (A2·A1, A2·U1+U2); left operand = later (Q2)."""
    assert oracle.compose((2.0, 3.0), (5.0, 7.0)) == (10.0, 17.0)
    assert oracle.compose((5.0, 7.0), (2.0, 3.0)) == (10.0, 22.0)
    # applying e1 then e2 to a state equals applying e2⊕e1
    h = 1.5
    A, U = oracle.compose((2.0, 3.0), (5.0, 7.0))
    assert A * h + U == 2.0 * (5.0 * h + 7.0) + 3.0
    # identity (Q3)
    assert oracle.compose((1.0, 0.0), (5.0, 7.0)) == (5.0, 7.0)
    assert oracle.compose((5.0, 7.0), (1.0, 0.0)) == (5.0, 7.0)
    # (0, v) is a left zero: it annihilates everything earlier (sequence-head reset)
    assert oracle.compose((0.0, 4.0), (5.0, 7.0)) == (0.0, 4.0)


@pytest.mark.parametrize("m", [2, 3, 5, 8])
def test_every_bracketing_agrees(m):
    """BJ / P:90-95: brute force over every tree bracketing of m pairs (Catalan(m-1) trees,
    429 for m=8) in exact arithmetic: all equal, equal to the oracle's fold, and equal to the
    sequential loop's (prod a, h_last at h0=0)."""
    a = dyadic(RNG, m, denom=4, lo=-6, hi=6)
    u = dyadic(RNG, m, denom=4)
    pairs = [(Fraction(float(x)), Fraction(float(y))) for x, y in zip(a, u)]
    results = set(all_bracketings(pairs))
    n_trees = sum(1 for _ in all_bracketings(pairs))
    catalan = math.comb(2 * (m - 1), m - 1) // m
    assert n_trees == catalan
    assert len(results) == 1
    A_ref, U_ref = next(iter(results))
    A_tot, U_tot = oracle.fold_pairs(a, u)
    assert (Fraction(A_tot), Fraction(U_tot)) == (A_ref, U_ref)
    h, h_last = oracle.affine_scan(a[None], u[None], None)
    assert Fraction(h_last[0]) == U_ref
    assert Fraction(float(np.prod(a))) == A_ref
    # and through oracle.compose on a few explicit (non-left-fold) trees
    def tree(lo, hi, rng):
        if hi - lo == 1:
            return (float(a[lo]), float(u[lo]))
        s = rng.integers(lo + 1, hi)
        return oracle.compose(tree(s, hi, rng), tree(lo, s, rng))
    for _ in range(10):
        At, Ut = tree(0, m, RNG)
        assert (Fraction(At), Fraction(Ut)) == (A_ref, U_ref)


def test_h_last_is_total_composition_applied_to_h0():
    """BJ / P:93: h_last = A_tot·h0 + U_tot."""
    for L in (1, 5, 64):
        a = dyadic(RNG, L, denom=2, lo=-2, hi=2) if L <= 5 else RNG.uniform(0.5, 0.99, L)
        u = dyadic(RNG, L, denom=2) if L <= 5 else RNG.normal(size=L)
        h0 = 2.5
        A_tot, U_tot = oracle.fold_pairs(a, u)
        _, h_last = oracle.affine_scan(a[None], u[None], np.array([h0]))
        if L <= 5:
            assert h_last[0] == A_tot * h0 + U_tot
        else:
            assert h_last[0] == pytest.approx(A_tot * h0 + U_tot, rel=1e-13)
    assert oracle.fold_pairs(np.zeros(0), np.zeros(0)) == (1.0, 0.0)


def test_every_prefix_is_a_fold():
    """the prefix composition up to t reproduces h_t."""
    L = 9
    a = dyadic(RNG, L, denom=4, lo=-5, hi=5)
    u = dyadic(RNG, L, denom=4)
    h0 = -0.75
    h, _ = oracle.affine_scan(a[None], u[None], np.array([h0]))
    for t in range(L):
        A_t, U_t = oracle.fold_pairs(a[:t + 1], u[:t + 1])
        assert h[0, t] == A_t * h0 + U_t


def test_linearity_and_power_of_two_scaling():
    a = RNG.uniform(0.5, 0.99, size=(2, 50))
    u1, u2 = dyadic(RNG, (2, 50)), dyadic(RNG, (2, 50))
    g1, g2 = dyadic(RNG, 2), dyadic(RNG, 2)
    h1, _ = oracle.affine_scan(a, u1, g1)
    h2, _ = oracle.affine_scan(a, u2, g2)
    h12, _ = oracle.affine_scan(a, u1 + u2, g1 + g2)
    np.testing.assert_allclose(h12, h1 + h2, rtol=1e-12, atol=1e-12)
    hs, _ = oracle.affine_scan(a, 8.0 * u1, 8.0 * g1)
    assert np.array_equal(hs, 8.0 * h1)          # scaling by 2^k is exact


@pytest.mark.parametrize("m", [0, 1, 17, 63, 64])
def test_split_invariance(m):
    """scanning [0,L) equals scanning [0,m) then [m,L) with h0' = h_last."""
    L = 64
    a = RNG.uniform(0.5, 0.99, size=(3, L))
    u = RNG.normal(size=(3, L))
    h0 = RNG.normal(size=3)
    h, hl = oracle.affine_scan(a, u, h0)
    ha, hla = oracle.affine_scan(a[:, :m], u[:, :m], h0)
    hb, hlb = oracle.affine_scan(a[:, m:], u[:, m:], hla)
    assert np.array_equal(np.concatenate([ha, hb], axis=1), h)
    assert np.array_equal(hlb, hl)


def test_weighted_prefix_mapping():
    """P:272-274 Eq.(10): h_t = α_t h_{t-1} + β_t is the affine scan with a=α, u=β·1; through
    the selective oracle it is x=1, c=1 (N=1), with a = exp(Δ·A) = α, b = Δ·B = β."""
    L = 30
    alpha = RNG.uniform(0.5, 0.99, size=L)
    beta = RNG.normal(size=L)
    h, _ = oracle.affine_scan(alpha[None], beta[None], None)
    # selective form: pick Δ=1 so that A·Δ = log α is impossible per-t (A is per-channel);
    # instead use constant α: A = log α0, Δ = 1, B = β, x = 1, C = 1.
    a0 = 0.8
    y, hl = oracle.selective_scan_fwd(np.ones((1, 1, L)), np.ones((1, 1, L)),
                                      np.array([[math.log(a0)]]), beta[None, None, :],
                                      np.ones((1, 1, L)), None, None)
    href, _ = oracle.affine_scan(np.full((1, L), a0), beta[None], None)
    np.testing.assert_allclose(y[0, 0], href[0], rtol=1e-13, atol=1e-15)


# ------------------------------------------------------------------ selective oracle
def selective_closed_form(x, delta, A, B, C, D, h0):
    """Independent evaluation that never steps the recurrence: with S_t = Σ_{k≤t} Δ_k,
        h_t[d,n] = exp(A[d,n] S_t) h0 + Σ_{k≤t} exp(A[d,n] (S_t − S_k)) Δ_k B_k[n] x_k
    (Eq.(5) with a_i = exp(Δ_i A): products of exps become exps of sums), then
        y_t[d] = Σ_n C_t[n] h_t[d,n] + D[d] x_t[d]          (BJ).
    O(L²·N); numpy broadcasting; used on tiny shapes only."""
    batch, d_inner, L = x.shape
    N = A.shape[1]
    y = np.zeros((batch, d_inner, L))
    h_last = np.zeros((batch, d_inner, N))
    for b in range(batch):
        for d in range(d_inner):
            S = np.cumsum(delta[b, d])                                   # [L]
            diff = S[:, None] - S[None, :]                               # [t, k]
            mask = np.tril(np.ones((L, L)))                              # k ≤ t
            for n in range(N):
                w = np.exp(A[d, n] * diff) * mask                        # [t, k]
                drive = delta[b, d] * B[b, n] * x[b, d]                  # [k]
                h = w @ drive
                if h0 is not None:
                    h = h + np.exp(A[d, n] * S) * h0[b, d, n]
                y[b, d] += C[b, n] * h
                h_last[b, d, n] = h[-1]
            if D is not None:
                y[b, d] += D[d] * x[b, d]
    return y, h_last


def _small_selective(batch=2, d_inner=3, N=4, L=37, with_D=True, with_h0=True):
    x = RNG.normal(size=(batch, d_inner, L))
    delta = np.log1p(np.exp(RNG.normal(size=(batch, d_inner, L)) - 2.0))
    A = -np.exp(RNG.uniform(-1, 1, size=(d_inner, N)))
    B = RNG.normal(size=(batch, N, L))
    C = RNG.normal(size=(batch, N, L))
    D = RNG.normal(size=d_inner) if with_D else None
    h0 = RNG.normal(size=(batch, d_inner, N)) if with_h0 else None
    return x, delta, A, B, C, D, h0


@pytest.mark.parametrize("with_D,with_h0", [(True, True), (False, False), (True, False)])
def test_selective_vs_independent_closed_form(with_D, with_h0):
    """Distinct batch/d_inner/N/L so any transposed layout or swapped B/C index fails."""
    args = _small_selective(with_D=with_D, with_h0=with_h0)
    y, hl = oracle.selective_scan_fwd(*args)
    y_ref, hl_ref = selective_closed_form(*args)
    np.testing.assert_allclose(y, y_ref, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(hl, hl_ref, rtol=1e-11, atol=1e-12)


def test_selective_reduces_to_affine_scan():
    """BJ: N=1, C≡1, D=NULL ⇒ y equals affine_scan(a = exp(Δ·A), u = Δ·B·x)."""
    batch, d_inner, L = 2, 3, 50
    x, delta, A, B, C, _, h0 = _small_selective(batch, d_inner, 1, L)
    y, hl = oracle.selective_scan_fwd(x, delta, A, B, np.ones_like(C), None, h0)
    a = np.exp(delta * A[None, :, 0:1])                        # [b,d,L]
    u = (delta * B[:, 0:1, :]) * x
    h, h_last = oracle.affine_scan(a.reshape(-1, L), u.reshape(-1, L), h0.reshape(-1))
    np.testing.assert_allclose(y.reshape(-1, L), h, rtol=1e-14, atol=0)
    np.testing.assert_allclose(hl.reshape(-1), h_last, rtol=1e-14, atol=0)


def test_selective_delta_zero_holds_state():
    """Δ≡0 ⇒ a=1,u=0 ⇒ h_t ≡ h0 and y_t = Σ_n C_t[n] h0[n] + D x_t (exact on dyadics)."""
    batch, d_inner, N, L = 2, 2, 3, 9
    x = dyadic(RNG, (batch, d_inner, L))
    C = dyadic(RNG, (batch, N, L))
    B = dyadic(RNG, (batch, N, L))
    h0 = dyadic(RNG, (batch, d_inner, N))
    D = dyadic(RNG, d_inner)
    A = -np.ones((d_inner, N))
    y, hl = oracle.selective_scan_fwd(x, np.zeros_like(x), A, B, C, D, h0)
    ref = np.einsum("bnl,bdn->bdl", C, h0) + D[None, :, None] * x
    np.testing.assert_allclose(y, ref, rtol=0, atol=1e-15)
    assert np.array_equal(hl, h0)


def test_selective_A_to_zero_is_cumsum():
    """A→0⁻ with N=1, B=C=1 ⇒ y = cumsum(Δ·x) + D·x."""
    L = 40
    x = RNG.normal(size=(1, 2, L))
    delta = RNG.uniform(0.01, 0.5, size=(1, 2, L))
    D = np.array([0.5, -1.5])
    y, hl = oracle.selective_scan_fwd(x, delta, np.full((2, 1), -1e-300), np.ones((1, 1, L)),
                                      np.ones((1, 1, L)), D, None)
    ref = np.cumsum(delta * x, axis=2) + D[None, :, None] * x
    np.testing.assert_allclose(y, ref, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(hl[..., 0], np.cumsum(delta * x, axis=2)[..., -1], rtol=1e-13)


def test_selective_one_hot_C_reads_one_state():
    """C one-hot in n ⇒ y is that state's trajectory; B one-hot drives only that state."""
    batch, d_inner, N, L = 1, 2, 4, 25
    x, delta, A, B, C, _, _ = _small_selective(batch, d_inner, N, L)
    for n in range(N):
        Cn = np.zeros_like(C)
        Cn[:, n, :] = 1.0
        y, hl = oracle.selective_scan_fwd(x, delta, A, B, Cn, None, None)
        for d in range(d_inner):
            a = np.exp(delta[0, d] * A[d, n])
            u = delta[0, d] * B[0, n] * x[0, d]
            h, h_last = oracle.affine_scan(a[None], u[None], None)
            np.testing.assert_allclose(y[0, d], h[0], rtol=1e-14)
            assert hl[0, d, n] == pytest.approx(h_last[0], rel=1e-14)


def test_selective_split_invariance():
    x, delta, A, B, C, D, h0 = _small_selective(L=64)
    y, hl = oracle.selective_scan_fwd(x, delta, A, B, C, D, h0)
    m = 23
    y1, hl1 = oracle.selective_scan_fwd(x[..., :m], delta[..., :m], A, B[..., :m], C[..., :m], D, h0)
    y2, hl2 = oracle.selective_scan_fwd(x[..., m:], delta[..., m:], A, B[..., m:], C[..., m:], D, hl1)
    assert np.array_equal(np.concatenate([y1, y2], axis=2), y)
    assert np.array_equal(hl2, hl)


# ----------------------------------------------------------------- Blelloch CPU model
@pytest.mark.parametrize("L", [1, 2, 3, 4, 7, 8, 9, 31, 32, 33, 100])
def test_blelloch_model_equals_loop(L):
    """P:103-107 / P:163-167 (Q3, Q4, Q16): upsweep, root ← (1,0), downsweep, reconstruction
    reproduce the sequential loop — bit for bit on dyadic inputs (short L), to rounding else."""
    if L <= 12:
        a = dyadic(RNG, L, denom=4, lo=-5, hi=5)
        u = dyadic(RNG, L, denom=4)
    else:
        a = RNG.uniform(0.5, 0.99, size=L)
        u = RNG.normal(size=L)
    h0 = 0.75
    hb = oracle.blelloch_scan(a, u, h0)
    h, _ = oracle.affine_scan(a[None], u[None], np.array([h0]))
    if L <= 12:
        assert np.array_equal(hb, h[0])
    else:
        np.testing.assert_allclose(hb, h[0], rtol=1e-12, atol=1e-13)
