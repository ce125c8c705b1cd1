"""Pins of oracle/ozaki.py: the INT8-slice emulation of an FP64 product against exact rational
arithmetic and against what the mathematics fixes (slice ranges, exact reconstruction, the error bound and its scaling)."""
from fractions import Fraction

import numpy as np
import pytest

from oracle.ozaki import S_DEFAULT, W, emulated_matmul, error_bound, scale_exponents, split


def _exact_matmul(a, b):
    """A B in exact rational arithmetic (every double is a dyadic rational), rounded to double once at the end."""
    fa = [[Fraction(float(x)) for x in row] for row in a]
    fb = [[Fraction(float(x)) for x in row] for row in b]
    out = np.zeros((len(fa), len(fb[0])))
    for i in range(len(fa)):
        for j in range(len(fb[0])):
            out[i, j] = float(sum(fa[i][l] * fb[l][j] for l in range(len(fb))))
    return out


def test_slices_are_int8_and_reconstruct_the_operand():
    rng = np.random.default_rng(0)
    a = rng.normal(size=(9, 33)) * np.exp(rng.normal(size=(9, 1)) * 8)          # rows of very different magnitude
    a[3] = 0.0                                                                    # a zero row
    a[5, :] = 2.0 ** -7                                                           # an exact power of two as the row maximum
    e, q = split(a, 1)
    assert q.dtype == np.int8 and q.shape == (S_DEFAULT,) + a.shape
    assert np.abs(q.astype(np.int64)).max() <= 127
    assert e[3] == 0 and (q[:, 3] == 0).all()
    v = np.ldexp(a, -e[:, None])
    assert (np.abs(v) < 1.0).all() and (np.abs(v).max(axis=1)[e != 0] >= 0.5).all()     # step 1 of the algorithm
    rec = sum(np.ldexp(q[s].astype(np.float64), -W * (s + 1)) for s in range(S_DEFAULT))
    assert np.abs(rec - v).max() < 2.0 ** (-W * S_DEFAULT)                       # |rho| < 2^(-WS)
    # truncation toward zero: every slice carries the sign of the value (or is zero)
    assert ((q.astype(np.int64) * np.sign(v)[None]) >= 0).all()
    # columns: the same along axis 0
    f, qb = split(a.T, 0)
    assert (f == e).all() and (qb == np.swapaxes(q, 1, 2)).all()
    assert list(scale_exponents(np.array([[1.0, 0.25], [0.75, 0.1], [2.0 ** -1074, 0.0]]), 1)) == [1, 0, -1073]


@pytest.mark.parametrize("m,k,n,seed", [(5, 7, 4, 1), (8, 16, 6, 2), (3, 64, 3, 3)])
def test_emulated_product_equals_exact_arithmetic_within_the_bound(m, k, n, seed):
    rng = np.random.default_rng(seed)
    a = rng.normal(size=(m, k)) * np.exp(rng.normal(size=(m, 1)) * 5)
    b = rng.normal(size=(k, n)) * np.exp(rng.normal(size=(1, n)) * 5)
    b[:, 0] = 0.0
    exact = _exact_matmul(a, b)
    got = emulated_matmul(a, b)
    bound = error_bound(a, b)
    assert (np.abs(got - exact) <= bound + 4 * np.finfo(float).eps * np.abs(exact)).all()
    assert (got[:, 0] == 0.0).all()
    # the bound is not vacuous: 49 bits is far below float64 rounding of the plain product for these sizes ...
    assert np.abs(got - exact).max() <= 1e-11 * np.abs(exact).max()
    # ... and lowering S loosens the error by 2^W per slice, as the analysis says
    errs = [np.abs(emulated_matmul(a, b, s) - exact).max() for s in (3, 4, 5)]
    assert errs[0] > 20 * errs[1] > 400 * errs[2] > 0
    for s in (3, 4, 5):
        assert (np.abs(emulated_matmul(a, b, s) - exact) <= error_bound(a, b, s)).all()


def test_emulated_product_at_microbenchmark_size_meets_the_parity_tolerance():
    """BASELINE.json configs[4] operands (N(0,1), 512-long contraction): error <= 1e-10 max|C| (the tolerance of north_star)
    with two decades of margin, against NumPy's FP64 product (itself accurate to ~1e-14 here)."""
    rng = np.random.default_rng(4)
    a, b = rng.normal(size=(96, 512)), rng.normal(size=(512, 80))
    ref = a @ b
    got = emulated_matmul(a, b)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    assert (np.abs(got - ref) <= error_bound(a, b) + 1e-13 * np.abs(ref).max()).all()
