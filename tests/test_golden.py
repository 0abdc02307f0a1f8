"""The stored expected values under tests/golden/ (written by tests/golden/make_golden.py from
oracle/ alone): the oracle reproduces them bit for bit, an exact-rational evaluation of Eq.(5)
agrees with them, and (GPU) every affine_scan variant matches them to 2 ulp."""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def read_golden(name):
    out = {}
    with open(os.path.join(HERE, "golden", name)) as f:
        lines = [ln for ln in f.read().splitlines() if ln and not ln.startswith("#")]
    i = 0
    while i < len(lines):
        key, r, c = lines[i].split()
        r, c = int(r), int(c)
        out[key] = np.array([[float.fromhex(v) for v in lines[i + 1 + j].split()] for j in range(r)])
        assert out[key].shape == (r, c)
        i += 1 + r
    return out


def test_oracle_reproduces_golden_bit_for_bit():
    g = read_golden("affine_dyadic.txt")
    h, h_last = oracle.affine_scan(g["a"], g["u"], g["h0"][0])
    assert np.array_equal(h, g["h"]) and np.array_equal(h_last, g["h_last"][0])


def test_golden_equals_exact_rational_closed_form():
    """PAPER.md Eq.(5) (line 81) in exact rational arithmetic: no floating point involved."""
    g = read_golden("affine_dyadic.txt")
    a, u, h0 = g["a"], g["u"], g["h0"][0]
    for s in range(a.shape[0]):
        for t in range(a.shape[1]):
            prod = Fraction(1)
            for i in range(t + 1):
                prod *= Fraction(a[s, i])
            tot = prod * Fraction(h0[s])
            for k in range(t + 1):
                w = Fraction(1)
                for i in range(k + 1, t + 1):
                    w *= Fraction(a[s, i])
                tot += w * Fraction(u[s, k])
            assert Fraction(g["h"][s, t]) == tot, (s, t)


@pytest.mark.gpu
def test_gpu_affine_variants_match_golden(cuda_device):
    import torch

    import paper_2606_00601_b200 as lib
    g = read_golden("affine_dyadic.txt")
    a = torch.tensor(g["a"], dtype=torch.float32, device=cuda_device)
    u = torch.tensor(g["u"], dtype=torch.float32, device=cuda_device)
    h0 = torch.tensor(g["h0"][0], dtype=torch.float32, device=cuda_device)
    for v in (lib.VARIANT_AUTO, lib.AFFINE_LOOKBACK, lib.AFFINE_CTA_LOOP, lib.AFFINE_WARP_SEQ,
              lib.AFFINE_BLELLOCH):
        h = torch.empty_like(a)
        hl = torch.empty(a.shape[0], dtype=torch.float32, device=cuda_device)
        lib.affine_scan_ex(a, u, h0, h, hl, v)
        torch.cuda.synchronize()
        # the stored values are fp32-representable; a tree bracketing may round an intermediate
        # pair in the last bit, so allow 2 ulp instead of demanding bitwise equality
        hh = h.cpu().numpy().astype(np.float64)
        assert np.max(np.abs(hh - g["h"]) / (1 + np.abs(g["h"]))) <= 2.4e-7, v
        assert np.max(np.abs(hl.cpu().numpy() - g["h_last"][0])) <= 2.4e-7 * 8, v
