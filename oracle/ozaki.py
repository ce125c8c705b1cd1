"""ORACLE (test infrastructure only; never imported by the product path).

FP64 matrix product emulated with exact integer products of INT8 slices ("Ozaki-style split into
INT8 slices with exact integer accumulation", the road past the FP64 ceiling the paper's headline is about, PAPER.md:7,
:255).  The paper gives no algorithm for it; this is the scheme the CUDA path (csrc/ozaki.cu) follows, written out step by
step in plain NumPy so that it can be checked by eye:

  1. scaling.  Row i of A gets the exponent e_i = floor(log2(max_j |a_ij|)) + 1, so that v_ij = a_ij 2^(-e_i) has |v| < 1
     (a zero row gets e_i = 0).  Columns of B likewise (f_j).
  2. slicing, S slices of W = 7 bits, by TRUNCATION toward zero: t = v 2^W; q_0 = trunc(t); t <- (t - q_0) 2^W; q_1 = trunc(t);
     ...  Every q_s is an integer in [-127, 127] (it fits INT8, and trunc never produces +-128 because |t| < 128), all
     operations are exact in binary floating point, and  v = sum_s q_s 2^(-W(s+1)) + rho,  |rho| < 2^(-W S).
  3. products.  For every pair (s, t) with s + t <= S - 1 the integer matrix product Q^A_s Q^B_t is EXACT in 32-bit
     integers as long as (d+1) k 127^2 < 2^31 for the diagonal sum below; pairs with s + t >= S are dropped (they are below
     the slicing error).
  4. diagonals.  P_d = sum_{s=0..d} Q^A_s Q^B_(d-s), d = 0..S-1, still exact integers (one GEMM over the concatenated
     contraction index of length (d+1) k: A slices in the order 0..d, B slices in the order d..0).
  5. recombination in FP64, smallest term first:  C_ij = 2^(e_i + f_j) sum_{d=S-1..0} P_d[i,j] 2^(-W(d+2)).

Error: |C - A B|_ij <= 2^(e_i + f_j) k (S + 2) 2^(-W S)  (dropped pairs + the two slicing remainders), i.e. relative to the
SCALE of row i and column j, not to |C_ij| itself -- the usual statement for this family of schemes.  With W = 7, S = 7
that is 9 k 2^(-49) 2^(e_i+f_j): 8e-12 of the scale product at k = 512.

Pins: tests/test_oracle_ozaki.py (slices are INT8 and reconstruct the operand to 2^(-WS); every P_d fits int32; the result
equals exact rational arithmetic within the bound on small integer-free cases; rows / columns of zeros and of wildly
different magnitude; the bound scales as stated when S is lowered).
"""
import numpy as np

W = 7          # bits per slice
S_DEFAULT = 7  # slices (49 bits)


def scale_exponents(a, axis):
    """e = floor(log2(max |a| along `axis`)) + 1 (0 for an all-zero line), kept as an integer array with that axis removed."""
    amax = np.max(np.abs(a), axis=axis)
    e = np.zeros(amax.shape, dtype=np.int64)
    nz = amax > 0
    e[nz] = np.floor(np.log2(amax[nz])).astype(np.int64) + 1
    # guard against log2 rounding at exact powers of two: enforce amax * 2^-e < 1 <= amax * 2^-(e-1)
    while True:
        v = np.ldexp(amax, -e)
        hi, lo = nz & (v >= 1.0), nz & (v < 0.5)
        if not hi.any() and not lo.any():
            return e
        e[hi] += 1
        e[lo] -= 1


def split(a, axis, nslices=S_DEFAULT):
    """Steps 1-2 for the lines of `a` that run along `axis` (axis = 1: rows of A; axis = 0: columns of B).
    Returns (e, q): exponents and the int8 slices q[s] (same shape as a)."""
    a = np.asarray(a, dtype=np.float64)
    e = scale_exponents(a, axis)
    t = np.ldexp(a, -np.expand_dims(e, axis))            # |t| < 1, exact
    q = np.zeros((nslices,) + a.shape, dtype=np.int8)
    for s in range(nslices):
        t = t * float(1 << W)                            # exact (power of two)
        qs = np.trunc(t)
        assert np.abs(qs).max(initial=0.0) <= 127.0
        q[s] = qs.astype(np.int8)
        t = t - qs                                       # exact: same binade or lower, |t| < 1
    return e, q


def emulated_matmul(a, b, nslices=S_DEFAULT):
    """Steps 1-5: C ~= A B (A: m x k, B: k x n) from exact integer slice products."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    k = a.shape[1]
    assert (nslices * k * 127 * 127) < 2 ** 31, "a diagonal would overflow 32-bit accumulation"
    e, qa = split(a, 1, nslices)
    f, qb = split(b, 0, nslices)
    c = np.zeros((a.shape[0], b.shape[1]))
    for d in range(nslices - 1, -1, -1):                 # smallest terms first
        p = np.zeros((a.shape[0], b.shape[1]), dtype=np.int64)
        for s in range(d + 1):
            p += qa[s].astype(np.int64) @ qb[d - s].astype(np.int64)
        assert np.abs(p).max(initial=0) < 2 ** 31        # what the INT8 tensor cores accumulate in
        c += np.ldexp(p.astype(np.float64), -W * (d + 2))
    return np.ldexp(c, e[:, None] + f[None, :])


def error_bound(a, b, nslices=S_DEFAULT):
    """Entry-wise bound of |emulated - exact| (docstring above)."""
    e = scale_exponents(np.asarray(a, dtype=np.float64), 1)
    f = scale_exponents(np.asarray(b, dtype=np.float64), 0)
    k = np.shape(a)[1]
    return np.ldexp(np.ones((len(e), len(f))), e[:, None] + f[None, :]) * k * (nslices + 2) * 2.0 ** (-W * nslices)
