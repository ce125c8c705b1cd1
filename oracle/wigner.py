"""ORACLE (test infrastructure only; never imported by the product path).

Wigner 6j / 9j symbols exactly as printed in PAPER.md Appendix A, Eqs. (9)-(15)
(PAPER.md:340-384), Clebsch-Gordan coefficients, and the SU(2) factor C-hat of
SURVEY.md section 8(c) C1.5 (the paper's Eq. (5)/(9), in
Wigner-Eckart convention "B").

All spin arguments are passed as DOUBLED integers (two_j = 2*j) so half-integers
are exact.  Everything is evaluated with exact integer factorials and converted to
float64 once at the end of each symbol.

Readings of garbled passages:
  G2  Eq. (11): x_min is printed without absolute values; we use
      x_min = max(|j1-j'|, |j2-k|, |k1-j2'|) (the triangle conditions of the three
      6j symbols); identical to the printed form whenever the printed form is valid.
  G3  Eq. (12): the six triads that must be triangular are
      (j1 j2 j), (k1 k2 k), (j1' j2' j'), (j1 k1 j1'), (j2 k2 j2'), (j k j').
  G4  Eq. (14): n~_1 = 0 only guards n_min >= 0.

Pins: tests/test_oracle_wigner.py (closed values, orthogonality, brute-force
Clebsch-Gordan sums, ladder-operator construction of coupled states).
"""
from fractions import Fraction
from functools import lru_cache
from math import factorial, sqrt


def _is_triad(a2, b2, c2):
    """|a-b| <= c <= a+b and a+b+c integer (doubled arguments)."""
    return (a2 + b2 + c2) % 2 == 0 and abs(a2 - b2) <= c2 <= a2 + b2


def _f(two_x):
    """factorial of an integer given as a doubled value."""
    assert two_x % 2 == 0 and two_x >= 0
    return factorial(two_x // 2)


def _g2(a2, b2, c2):
    """Square of the paper's g~(a,b,c), Eq. (15), as an exact Fraction."""
    return Fraction(_f(a2 + b2 - c2) * _f(a2 - b2 + c2) * _f(-a2 + b2 + c2), _f(a2 + b2 + c2 + 2))


@lru_cache(maxsize=None)
def w6j(a2, b2, c2, d2, e2, f2):
    """W6j(a,b,c,d,e,f) of Eq. (13)-(15): the standard 6j symbol
    {a b c; d e f} as a Racah sum.  Returns 0.0 outside the triangle rules of Eq. (14)."""
    if not (_is_triad(a2, b2, c2) and _is_triad(c2, d2, e2) and _is_triad(a2, e2, f2) and _is_triad(b2, d2, f2)):
        return 0.0
    n2 = a2 + b2 + c2
    n3 = c2 + d2 + e2
    n4 = a2 + e2 + f2
    n5 = b2 + d2 + f2
    n6 = a2 + b2 + d2 + e2
    n7 = a2 + c2 + d2 + f2
    n8 = b2 + c2 + e2 + f2
    nmin = max(0, n2, n3, n4, n5)
    nmax = min(n6, n7, n8)
    s = Fraction(0)
    for n in range(nmin, nmax + 1, 2):          # doubled n; all n~ are even (integers)
        den = _f(n - n2) * _f(n - n3) * _f(n - n4) * _f(n - n5) * _f(n6 - n) * _f(n7 - n) * _f(n8 - n)
        s += Fraction((-1) ** (n // 2) * _f(n + 2), den)
    pref2 = _g2(a2, b2, c2) * _g2(c2, d2, e2) * _g2(a2, e2, f2) * _g2(b2, d2, f2)
    return float(s) * sqrt(pref2.numerator) / sqrt(pref2.denominator)


@lru_cache(maxsize=None)
def w9j(j1, j2, j, k1, k2, k, j1p, j2p, jp):
    """W9j(j1,j2,j,k1,k2,k,j1',j2',j') of Eq. (10)-(12): the 9j symbol
    with rows (j1 j2 j), (k1 k2 k), (j1' j2' j') as a sum over x of three 6j symbols."""
    triads = ((j1, j2, j), (k1, k2, k), (j1p, j2p, jp), (j1, k1, j1p), (j2, k2, j2p), (j, k, jp))
    if not all(_is_triad(*t) for t in triads):
        return 0.0
    xmin = max(abs(j1 - jp), abs(j2 - k), abs(k1 - j2p))
    xmax = min(j1 + jp, j2 + k, k1 + j2p)
    s = 0.0
    for x in range(xmin, xmax + 1, 2):
        s += (-1) ** x * (x + 1) * w6j(j1, j2, j, k, jp, x) * w6j(k1, k2, k, j2, x, j2p) * w6j(j1p, j2p, jp, x, j1, k1)
    return s


@lru_cache(maxsize=None)
def cg(j1, m1, j2, m2, j, m):
    """Clebsch-Gordan <j1 m1; j2 m2 | j m> (Condon-Shortley phases), textbook Racah
    formula; the paper only remarks that 6j/9j follow from these."""
    if m1 + m2 != m or not _is_triad(j1, j2, j):
        return 0.0
    if abs(m1) > j1 or abs(m2) > j2 or abs(m) > j:
        return 0.0
    if (j1 + m1) % 2 or (j2 + m2) % 2 or (j + m) % 2:
        return 0.0
    pref2 = Fraction((j + 1) * _f(j + j1 - j2) * _f(j - j1 + j2) * _f(j1 + j2 - j), _f(j1 + j2 + j + 2))
    pref2 *= _f(j + m) * _f(j - m) * _f(j1 - m1) * _f(j1 + m1) * _f(j2 - m2) * _f(j2 + m2)
    s = Fraction(0)
    kmin = max(0, j2 - j - m1, j1 + m2 - j)
    kmax = min(j1 + j2 - j, j1 - m1, j2 + m2)
    for kk in range(kmin, kmax + 1, 2):
        den = _f(kk) * _f(j1 + j2 - j - kk) * _f(j1 - m1 - kk) * _f(j2 + m2 - kk) * _f(j - j2 + m1 + kk) * _f(j - j1 - m2 + kk)
        s += Fraction((-1) ** (kk // 2), den)
    return float(s) * sqrt(pref2.numerator) / sqrt(pref2.denominator)


def c_hat(j1, j2, j, k1, k2, k, j1p, j2p, jp):
    """C-hat(j1,j2,j | k1,k2,k | j1',j2',j') = sqrt((2j1+1)(2j2+1)(2j'+1)(2k+1)) * W9j(...)
    (SURVEY.md 8(c) C1.5): the paper's Eq. (5) with its prefactor rewritten for the
    Wigner-Eckart convention <j m|T^k_q|j' m'> = <k q; j' m'|j m> <j||T||j'> used here."""
    return sqrt((j1 + 1) * (j2 + 1) * (jp + 1) * (k + 1)) * w9j(j1, j2, j, k1, k2, k, j1p, j2p, jp)


def c_tilde_paper(j1, j2, j, k1, k2, k, j1p, j2p, jp):
    """Eq. (5)/(9) exactly as printed; valid in the mirrored
    convention <j m|T^k_q|j' m'> = <j m; k q|j' m'> <j||T||j'>."""
    return sqrt((j1p + 1) * (j2p + 1) * (j + 1) * (k + 1)) * w9j(j1, j2, j, k1, k2, k, j1p, j2p, jp)
