"""Pins for the oracle's extended forward (softplus/bias prologue, silu(z) gate, resets: SURVEY
§8f-1/f-2) and for its backward pass (§8f-3), against things that are NOT
those functions: the already pinned plain forward oracle, math-library closed forms, hand
derivatives of a one-step problem and central finite differences.  CPU only.
"""
import math

import numpy as np
import pytest

import oracle

RNG = np.random.default_rng(20260603)


def _small(batch=2, d_inner=3, N=4, L=29, with_D=True, with_h0=True):
    x = RNG.normal(size=(batch, d_inner, L))
    delta = np.log1p(np.exp(RNG.normal(size=(batch, d_inner, L)) - 2.0))
    A = -np.exp(RNG.uniform(-1, 1, size=(d_inner, N)))
    B = RNG.normal(size=(batch, N, L))
    C = RNG.normal(size=(batch, N, L))
    D = RNG.normal(size=d_inner) if with_D else None
    h0 = RNG.normal(size=(batch, d_inner, N)) if with_h0 else None
    return x, delta, A, B, C, D, h0


# ------------------------------------------------------------------ extended forward
def test_ext_with_every_option_off_is_the_plain_forward_bitwise():
    x, delta, A, B, C, D, h0 = _small()
    y0, hl0 = oracle.selective_scan_fwd(x, delta, A, B, C, D, h0)
    y1, hl1 = oracle.selective_scan_fwd_ext(x, delta, A, B, C, D, None, None, None, h0, False)
    assert np.array_equal(y0, y1) and np.array_equal(hl0, hl1)
    # an all-zero reset mask and a zero bias change nothing either
    y2, hl2 = oracle.selective_scan_fwd_ext(x, delta, A, B, C, D, None, np.zeros(3),
                                            np.zeros((2, 29)), h0, False)
    assert np.array_equal(y0, y2) and np.array_equal(hl0, hl2)


def test_softplus_prologue_against_its_inverse_and_the_math_library():
    """Delta_raw = log(expm1(Delta)) - bias  =>  softplus(Delta_raw + bias) = Delta, so the
    extended call reproduces the plain forward on Delta (to rounding of the inverse)."""
    x, delta, A, B, C, D, h0 = _small()
    bias = RNG.normal(size=3)
    raw = np.log(np.expm1(delta)) - bias[None, :, None]
    y0, hl0 = oracle.selective_scan_fwd(x, delta, A, B, C, D, h0)
    y1, hl1 = oracle.selective_scan_fwd_ext(x, raw, A, B, C, D, None, bias, None, h0, True)
    np.testing.assert_allclose(y1, y0, rtol=1e-11, atol=1e-11)
    np.testing.assert_allclose(hl1, hl0, rtol=1e-11, atol=1e-11)
    # the bias alone (no softplus) is a plain shift: Delta = raw + bias
    y2, _ = oracle.selective_scan_fwd_ext(x, delta - bias[None, :, None], A, B, C, D, None, bias,
                                          None, h0, False)
    np.testing.assert_allclose(y2, y0, rtol=1e-12, atol=1e-12)
    # large arguments: softplus(v) -> v (no overflow); very negative: -> exp(v)
    one = np.ones((1, 1, 1))
    A1, B1, C1 = -np.ones((1, 1)), np.ones((1, 1, 1)), np.ones((1, 1, 1))
    for v in (800.0, 40.0, 0.0, -3.0, -50.0):
        yv, _ = oracle.selective_scan_fwd_ext(one, v * one, A1, B1, C1, None, None, None, None,
                                              None, True)
        sp = v + math.log1p(math.exp(-v)) if v > 0 else math.log1p(math.exp(v))
        assert yv[0, 0, 0] == pytest.approx(sp, rel=1e-14)      # y = Delta*B*x with h0 = 0


def test_bias_to_minus_infinity_holds_the_state():
    """softplus(raw + bias) -> 0 as bias -> -inf: a = 1, u = 0, so h_t = h0 and
    y_t = C_t . h0 + D x_t (the delta == 0 pin of the plain oracle, reached through the bias)."""
    x, delta, A, B, C, D, h0 = _small()
    y, hl = oracle.selective_scan_fwd_ext(x, delta, A, B, C, D, None, np.full(3, -800.0), None,
                                          h0, True)
    ref = np.einsum("bnl,bdn->bdl", C, h0) + D[None, :, None] * x
    np.testing.assert_allclose(y, ref, rtol=1e-13, atol=1e-13)
    np.testing.assert_array_equal(hl, h0)


def test_silu_gate_closed_form_and_limits():
    x, delta, A, B, C, D, h0 = _small()
    z = RNG.normal(size=x.shape) * 3
    y0, hl0 = oracle.selective_scan_fwd(x, delta, A, B, C, D, h0)
    y1, hl1 = oracle.selective_scan_fwd_ext(x, delta, A, B, C, D, z, None, None, h0, False)
    silu = np.vectorize(lambda v: v / (1.0 + math.exp(-v)))(z)
    np.testing.assert_allclose(y1, y0 * silu, rtol=1e-14, atol=0)
    assert np.array_equal(hl1, hl0)                      # the gate never touches the state
    # silu(0) = 0 kills y; z -> +large: silu(z) -> z; z -> -large: silu(z) -> 0
    yz, _ = oracle.selective_scan_fwd_ext(x, delta, A, B, C, D, np.zeros_like(x), None, None, h0)
    assert np.all(yz == 0.0)
    yb, _ = oracle.selective_scan_fwd_ext(x, delta, A, B, C, D, np.full_like(x, 50.0), None, None, h0)
    np.testing.assert_allclose(yb, 50.0 * y0, rtol=1e-15)
    yn, _ = oracle.selective_scan_fwd_ext(x, delta, A, B, C, D, np.full_like(x, -700.0), None, None, h0)
    assert np.max(np.abs(yn)) < 1e-290


@pytest.mark.parametrize("cuts", [(0,), (1,), (13,), (28,), (5, 6, 20)])
def test_reset_equals_independent_calls_split_at_the_reset(cuts):
    """A reset at t makes step t the left-zero pair (0, u_t): the packed call equals
    independent calls on the pieces, each piece after the first starting from h = 0 (split
    invariance of the plain oracle, in reverse).  Batch 1 resets at `cuts`, batch 0 never."""
    x, delta, A, B, C, D, h0 = _small()
    L = x.shape[2]
    reset = np.zeros((2, L))
    for c in cuts:
        reset[1, c] = 1.0
    y, hl = oracle.selective_scan_fwd_ext(x, delta, A, B, C, D, None, None, reset, h0, False)
    # batch 0: untouched
    y0, hl0 = oracle.selective_scan_fwd(x[:1], delta[:1], A, B[:1], C[:1], D, h0[:1])
    assert np.array_equal(y[:1], y0) and np.array_equal(hl[:1], hl0)
    # batch 1: pieces
    edges = [0] + [c for c in cuts if c > 0] + [L]
    carry = None if 0 in cuts else h0[1:]               # a reset at t = 0 discards h0
    for lo, hi in zip(edges[:-1], edges[1:]):
        yp, hp = oracle.selective_scan_fwd(x[1:, :, lo:hi], delta[1:, :, lo:hi], A,
                                           B[1:, :, lo:hi], C[1:, :, lo:hi], D, carry)
        assert np.array_equal(y[1:, :, lo:hi], yp)
        carry = None                                     # the next piece starts from zero
    assert np.array_equal(hl[1:], hp)


# ------------------------------------------------------------------------- backward
def test_backward_one_step_hand_derivatives():
    """N = 1, L = 1: y = C (exp(Delta A) h0 + Delta B x) + D x; derivatives written by hand."""
    xs, dl, A, B, C, D, h0, dy, dhl = 0.7, 0.3, -1.3, 0.9, -0.4, 1.7, 0.6, 2.5, -0.8
    a = math.exp(dl * A)
    g = C * dy + dhl                                      # d loss / d h_0step
    out = oracle.selective_scan_bwd(np.full((1, 1, 1), xs), np.full((1, 1, 1), dl),
                                    np.full((1, 1), A), np.full((1, 1, 1), B),
                                    np.full((1, 1, 1), C), np.full(1, D), np.full((1, 1, 1), h0),
                                    np.full((1, 1, 1), dy), np.full((1, 1, 1), dhl))
    h = a * h0 + dl * B * xs
    assert out["dx"].item() == pytest.approx(g * dl * B + D * dy, rel=1e-14)
    assert out["ddelta"].item() == pytest.approx(g * (A * a * h0 + B * xs), rel=1e-14)
    assert out["dA"].item() == pytest.approx(g * dl * a * h0, rel=1e-14)
    assert out["dB"].item() == pytest.approx(g * dl * xs, rel=1e-14)
    assert out["dC"].item() == pytest.approx(dy * h, rel=1e-14)
    assert out["dD"].item() == pytest.approx(dy * xs, rel=1e-14)
    assert out["dh0"].item() == pytest.approx(g * a, rel=1e-14)


def _loss(args, dy, dhl):
    y, hl = oracle.selective_scan_fwd(*args)
    return float(np.sum(dy * y) + np.sum(dhl * hl))


@pytest.mark.parametrize("with_D,with_h0", [(True, True), (False, False)])
def test_backward_against_central_finite_differences(with_D, with_h0):
    """Every entry of every gradient against (loss(v + e) - loss(v - e)) / 2e of the pinned
    forward oracle (float64, e = 1e-6: truncation ~1e-10, rounding ~1e-9)."""
    args = list(_small(batch=2, d_inner=2, N=3, L=11, with_D=with_D, with_h0=with_h0))
    dy = RNG.normal(size=args[0].shape)
    dhl = RNG.normal(size=(2, 2, 3))
    out = oracle.selective_scan_bwd(*args, dy, dhl)
    names = ["dx", "ddelta", "dA", "dB", "dC", "dD", "dh0"]
    eps = 1e-6
    for idx, name in enumerate(names):
        v = args[idx]
        if v is None:
            continue
        num = np.zeros_like(v)
        it = np.nditer(v, flags=["multi_index"])
        for _ in it:
            i = it.multi_index
            keep = v[i]
            v[i] = keep + eps
            lp = _loss(args, dy, dhl)
            v[i] = keep - eps
            lm = _loss(args, dy, dhl)
            v[i] = keep
            num[i] = (lp - lm) / (2 * eps)
        np.testing.assert_allclose(out[name], num, rtol=2e-6, atol=2e-7, err_msg=name)


def test_backward_adjoint_identity_and_linearity_in_dy():
    """<dy, J v> = <J^T dy, v> for the x-direction (y is affine in x at fixed Delta, so a plain
    difference gives J v exactly up to rounding); gradients are linear in (dy, dh_last)."""
    args = list(_small(batch=1, d_inner=3, N=4, L=40))
    x = args[0]
    v = RNG.normal(size=x.shape)
    dy = RNG.normal(size=x.shape)
    y0, _ = oracle.selective_scan_fwd(*args)
    args_v = [x + v] + args[1:]
    y1, _ = oracle.selective_scan_fwd(*args_v)
    out = oracle.selective_scan_bwd(*args, dy, None)
    assert np.sum(dy * (y1 - y0)) == pytest.approx(np.sum(out["dx"] * v), rel=1e-10)
    out2 = oracle.selective_scan_bwd(*args, 2.0 * dy, None)
    for k in out:
        np.testing.assert_allclose(out2[k], 2.0 * out[k], rtol=1e-14, atol=0)


def test_backward_sums_shared_parameters_over_rows_and_batches():
    """dB, dC sum over d; dA, dD sum over batch: splitting the rows and adding the parts gives
    the whole (catches a missing or doubled accumulation)."""
    x, delta, A, B, C, D, h0 = _small(batch=2, d_inner=4, N=3, L=17)
    dy = RNG.normal(size=x.shape)
    whole = oracle.selective_scan_bwd(x, delta, A, B, C, D, h0, dy, None)
    parts = [oracle.selective_scan_bwd(x[:, s], delta[:, s], A[s], B, C, D[s], h0[:, s], dy[:, s], None)
             for s in (slice(0, 1), slice(1, 4))]
    np.testing.assert_allclose(whole["dB"], parts[0]["dB"] + parts[1]["dB"], rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(whole["dC"], parts[0]["dC"] + parts[1]["dC"], rtol=1e-12, atol=1e-13)
    bparts = [oracle.selective_scan_bwd(x[b:b + 1], delta[b:b + 1], A, B[b:b + 1], C[b:b + 1], D,
                                        h0[b:b + 1], dy[b:b + 1], None) for b in range(2)]
    np.testing.assert_allclose(whole["dA"], bparts[0]["dA"] + bparts[1]["dA"], rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(whole["dD"], bparts[0]["dD"] + bparts[1]["dD"], rtol=1e-12, atol=1e-13)
