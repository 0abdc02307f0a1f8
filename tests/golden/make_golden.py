#!/usr/bin/env python
"""Writes tests/golden/*.txt.  Calls ONLY oracle/ (never the CUDA path).

The paper (arxiv/paper_2606_00601) prints no worked numeric example, so these files do not pin
the oracle to the paper; they freeze the oracle's output on tiny dyadic-rational inputs whose
results are exact in float64 (so any platform must reproduce them bit for bit), after the
oracle itself has passed its mathematical pins (tests/test_oracle_pins.py).  The GPU parity
tests also read them: a second, stored route from PAPER.md Eq.(3)/(5)-(7) to expected values.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
import oracle  # noqa: E402


def affine_case():
    # a in {k/8}, u small integers, h0 integer: every product/sum is exact in binary64
    # (Eq.3, h0 from P:81 Eq.5)
    a = np.array([[4, 2, 6, 1, 8, 3, 5, 7, 0, 4, 2, 6],
                  [8, 8, 8, 8, 4, 4, 4, 4, 2, 2, 2, 2]], dtype=np.float64) / 8.0
    u = np.array([[1, -2, 3, 0, 5, -1, 2, 2, 7, -3, 1, 4],
                  [1, 1, 1, 1, -1, -1, -1, -1, 2, 2, 2, 2]], dtype=np.float64)
    h0 = np.array([3.0, -2.0])
    h, h_last = oracle.affine_scan(a, u, h0)
    return a, u, h0, h, h_last


def write_matrix(f, name, m):
    m = np.atleast_2d(np.asarray(m, dtype=np.float64))
    f.write(f"{name} {m.shape[0]} {m.shape[1]}\n")
    for row in m:
        f.write(" ".join(float(v).hex() for v in row) + "\n")


def main():
    a, u, h0, h, h_last = affine_case()
    with open(os.path.join(HERE, "affine_dyadic.txt"), "w") as f:
        f.write("# affine_scan on dyadic rationals; written by tests/golden/make_golden.py from oracle/\n")
        f.write("# recurrence h_t = a_t h_{t-1} + u_t: PAPER.md line 69 (Eq.3), h_0: line 81 (Eq.5)\n")
        f.write("# values are C99 hex floats (exact)\n")
        for name, m in (("a", a), ("u", u), ("h0", h0), ("h", h), ("h_last", h_last)):
            write_matrix(f, name, m)
    print("wrote affine_dyadic.txt")


if __name__ == "__main__":
    main()
