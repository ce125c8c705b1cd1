"""Pins P1, P2, P5 for oracle/wigner.py (Eqs. (5), (9)-(15))."""
import itertools
import random
from math import sqrt

import numpy as np
import pytest

from conftest import golden_lines
from oracle.wigner import c_hat, c_tilde_paper, cg, w6j, w9j


def _tri(a, b, c):
    return (a + b + c) % 2 == 0 and abs(a - b) <= c <= a + b


def test_golden_closed_values():
    for p in golden_lines("wigner_values.txt"):
        n = 6 if p[0] == "6j" else 9
        args = [int(x) for x in p[1:1 + n]]
        val = eval(" ".join(p[1 + n:]))
        got = (w6j if p[0] == "6j" else w9j)(*args)
        assert abs(got - val) < 1e-14, (p, got)


def test_cg_textbook_values_and_orthogonality():
    s2, s3 = sqrt(2.0), sqrt(3.0)
    assert abs(cg(1, 1, 1, -1, 2, 0) - 1 / s2) < 1e-15
    assert abs(cg(1, 1, 1, -1, 0, 0) - 1 / s2) < 1e-15
    assert abs(cg(1, -1, 1, 1, 0, 0) + 1 / s2) < 1e-15
    assert abs(cg(2, 2, 2, -2, 0, 0) - 1 / s3) < 1e-15
    assert abs(cg(2, 0, 2, 0, 0, 0) + 1 / s3) < 1e-15
    assert abs(cg(2, 0, 2, 0, 4, 0) - sqrt(2.0 / 3.0)) < 1e-15
    assert abs(cg(2, 2, 1, -1, 1, 1) - sqrt(2.0 / 3.0)) < 1e-15
    assert abs(cg(2, 0, 1, 1, 1, 1) + sqrt(1.0 / 3.0)) < 1e-15
    for j1, j2 in itertools.product(range(0, 5), repeat=2):
        for j in range(abs(j1 - j2), j1 + j2 + 1, 2):
            for jp in range(abs(j1 - j2), j1 + j2 + 1, 2):
                for m in range(-min(j, jp), min(j, jp) + 1, 2):
                    s = sum(cg(j1, m1, j2, m - m1, j, m) * cg(j1, m1, j2, m - m1, jp, m) for m1 in range(-j1, j1 + 1, 2))
                    assert abs(s - (1.0 if j == jp else 0.0)) < 1e-13


def test_cg_matches_ladder_construction():
    """Coupled states built by diagonalising (J1+J2)^2 and stepping down with J_-:
    independent of the Racah formula (fixes magnitudes and Condon-Shortley phases)."""
    def spin_mats(two_j):
        d = two_j + 1
        ms = [two_j / 2 - i for i in range(d)]
        jz = np.diag(ms)
        jm = np.zeros((d, d))
        for i in range(d - 1):
            m = ms[i]
            jm[i + 1, i] = sqrt((two_j / 2 + m) * (two_j / 2 - m + 1))
        return jz, jm

    for j1, j2 in [(1, 1), (2, 1), (3, 2), (4, 3), (2, 2)]:
        z1, m1 = spin_mats(j1)
        z2, m2 = spin_mats(j2)
        e1, e2 = np.eye(j1 + 1), np.eye(j2 + 1)
        jz = np.kron(z1, e2) + np.kron(e1, z2)
        jm = np.kron(m1, e2) + np.kron(e1, m2)
        for j in range(abs(j1 - j2), j1 + j2 + 1, 2):
            # highest weight |j j>: orthogonal to all |j' j> with j' > j, positive <j1 j1; j2 (j-j1)|
            vec = np.array([cg(j1, j1 - 2 * a, j2, j2 - 2 * b, j, j) for a in range(j1 + 1) for b in range(j2 + 1)])
            assert abs(np.linalg.norm(vec) - 1) < 1e-13
            assert np.abs(jm.T @ vec).max() < 1e-12                     # J_+ |j j> = 0
            first = next(x for x in vec if abs(x) > 1e-12)
            assert first > 0                                            # Condon-Shortley: <j1 j1; j2 j-j1|j j> > 0
            cur, m = vec, j
            while m > -j:
                nxt = jm @ cur / sqrt((j / 2 + m / 2) * (j / 2 - m / 2 + 1))
                m -= 2
                ref = np.array([cg(j1, j1 - 2 * a, j2, j2 - 2 * b, j, m) for a in range(j1 + 1) for b in range(j2 + 1)])
                assert np.abs(nxt - ref).max() < 1e-12
                cur = nxt


def _six_j_from_cg(a, b, c, d, e, f):
    """Definition of the 6j symbol as the recoupling coefficient
    <(ab)c,d;e|a,(bd)f;e> = (-1)^(a+b+d+e) sqrt((2c+1)(2f+1)) {a b c; d e f}."""
    tot = 0.0
    me = e
    for ma in range(-a, a + 1, 2):
        for mb in range(-b, b + 1, 2):
            md = me - ma - mb
            if abs(md) > d:
                continue
            tot += (cg(a, ma, b, mb, c, ma + mb) * cg(c, ma + mb, d, md, e, me)
                    * cg(b, mb, d, md, f, mb + md) * cg(a, ma, f, mb + md, e, me))
    return tot * (-1) ** ((a + b + d + e) // 2) / sqrt((c + 1) * (f + 1))


def test_6j_equals_recoupling_definition_and_orthogonality():
    rng = range(0, 5)
    n = 0
    for a, b, c, d, e, f in itertools.product(rng, repeat=6):
        if _tri(a, b, c) and _tri(c, d, e) and _tri(a, e, f) and _tri(b, d, f):
            assert abs(w6j(a, b, c, d, e, f) - _six_j_from_cg(a, b, c, d, e, f)) < 1e-13
            n += 1
        else:
            assert w6j(a, b, c, d, e, f) == 0.0
    assert n > 300
    # orthogonality sum_x (2x+1) {a b x; d e c}{a b x; d e c'} = delta_cc'/(2c+1)   (P1)
    a, b, d, e = 2, 1, 3, 2
    for c in range(0, 7):
        for cp in range(0, 7):
            if not (_tri(a, e, c) and _tri(b, d, c) and _tri(a, e, cp) and _tri(b, d, cp)):
                continue
            s = sum((x + 1) * w6j(a, b, x, d, e, c) * w6j(a, b, x, d, e, cp) for x in range(0, 8))
            assert abs(s - (1.0 / (c + 1) if c == cp else 0.0)) < 1e-13


def _c_hat_brute(j1, j2, j, k1, k2, k, j1p, j2p, jp):
    """<(j1 j2)j||[T x U]^k||(j1' j2')j'> with unit reduced elements of T and U, straight from
    Clebsch-Gordan sums and the Wigner-Eckart convention B."""
    for m in range(-j, j + 1, 2):
        for q in range(-k, k + 1, 2):
            mp = m - q
            den = cg(k, q, jp, mp, j, m)
            if abs(den) < 1e-6:
                continue
            tot = 0.0
            for m1 in range(-j1, j1 + 1, 2):
                m2 = m - m1
                if abs(m2) > j2:
                    continue
                for q1 in range(-k1, k1 + 1, 2):
                    q2 = q - q1
                    if abs(q2) > k2:
                        continue
                    m1p, m2p = m1 - q1, m2 - q2
                    if abs(m1p) > j1p or abs(m2p) > j2p:
                        continue
                    tot += (cg(j1, m1, j2, m2, j, m) * cg(k1, q1, k2, q2, k, q) * cg(j1p, m1p, j2p, m2p, jp, mp)
                            * cg(k1, q1, j1p, m1p, j1, m1) * cg(k2, q2, j2p, m2p, j2, m2))
            return tot / den
    return 0.0


def test_c_hat_and_9j_against_brute_force_cg():
    """P2/P5: the SU(2) factor of Eq. (5)/(9) in convention B."""
    rnd = random.Random(7)
    done = 0
    while done < 250:
        j1, j2, j1p, j2p = (rnd.randrange(0, 4) for _ in range(4))
        k1, k2 = rnd.randrange(0, 3), rnd.randrange(0, 3)
        j = rnd.choice(range(abs(j1 - j2), j1 + j2 + 1, 2))
        jp = rnd.choice(range(abs(j1p - j2p), j1p + j2p + 1, 2))
        k = rnd.choice(range(abs(k1 - k2), k1 + k2 + 1, 2))
        if not (_tri(j1, k1, j1p) and _tri(j2, k2, j2p) and _tri(j, k, jp)):
            continue
        ref = _c_hat_brute(j1, j2, j, k1, k2, k, j1p, j2p, jp)
        assert abs(c_hat(j1, j2, j, k1, k2, k, j1p, j2p, jp) - ref) < 1e-12
        done += 1


def _el_mirrored(j, m, k, q, jp, mp):
    """Matrix element of a unit-reduced tensor operator in the MIRRORED Wigner-Eckart convention (bra and operator
    couple to the ket): <j m|T^k_q|j' m'> = (-1)^(k-q) <j m; k -q|j' m'> <j||T||j'>  (reading G1)."""
    return (-1) ** ((k - q) // 2) * cg(j, m, k, -q, jp, mp)


def _c_tilde_brute_mirrored(j1, j2, j, k1, k2, k, j1p, j2p, jp):
    """<(j1 j2)j||[T x U]^k||(j1' j2')j'> with unit reduced elements, from Clebsch-Gordan sums only, every
    Wigner-Eckart step taken in the mirrored convention of _el_mirrored."""
    for m in range(-j, j + 1, 2):
        for q in range(-k, k + 1, 2):
            mp = m - q
            if abs(mp) > jp:
                continue
            den = _el_mirrored(j, m, k, q, jp, mp)
            if abs(den) < 1e-6:
                continue
            tot = 0.0
            for m1 in range(-j1, j1 + 1, 2):
                m2 = m - m1
                if abs(m2) > j2:
                    continue
                for q1 in range(-k1, k1 + 1, 2):
                    q2 = q - q1
                    if abs(q2) > k2:
                        continue
                    m1p, m2p = m1 - q1, m2 - q2
                    if abs(m1p) > j1p or abs(m2p) > j2p:
                        continue
                    tot += (cg(j1, m1, j2, m2, j, m) * cg(k1, q1, k2, q2, k, q) * cg(j1p, m1p, j2p, m2p, jp, mp)
                            * _el_mirrored(j1, m1, k1, q1, j1p, m1p) * _el_mirrored(j2, m2, k2, q2, j2p, m2p))
            return tot / den
    return 0.0


def test_printed_prefactor_is_the_mirrored_convention():
    """G1: Eq. (5)/(9) exactly as printed (prefactor sqrt((2j1'+1)(2j2'+1)(2j+1)(2k+1))) is the
    product formula of the mirrored Wigner-Eckart convention -- brute-force Clebsch-Gordan sums, no 6j/9j on the
    reference side -- and it is NOT the formula of the convention the code uses (where c_hat holds)."""
    rnd = random.Random(11)
    done = differs = 0
    while done < 250:
        j1, j2, j1p, j2p = (rnd.randrange(0, 4) for _ in range(4))
        k1, k2 = rnd.randrange(0, 3), rnd.randrange(0, 3)
        j = rnd.choice(range(abs(j1 - j2), j1 + j2 + 1, 2))
        jp = rnd.choice(range(abs(j1p - j2p), j1p + j2p + 1, 2))
        k = rnd.choice(range(abs(k1 - k2), k1 + k2 + 1, 2))
        if not (_tri(j1, k1, j1p) and _tri(j2, k2, j2p) and _tri(j, k, jp)):
            continue
        ref = _c_tilde_brute_mirrored(j1, j2, j, k1, k2, k, j1p, j2p, jp)
        got = c_tilde_paper(j1, j2, j, k1, k2, k, j1p, j2p, jp)
        assert abs(got - ref) < 1e-12
        differs += abs(got - _c_hat_brute(j1, j2, j, k1, k2, k, j1p, j2p, jp)) > 1e-6
        done += 1
    assert differs > 50          # the two conventions really differ: the printed form must not be mixed with B


def test_9j_orthogonality_and_k0_reduction():
    # sum_{c,f} (2c+1)(2f+1)(2g+1)(2h+1) {abc;def;ghi}{abc;def;g'h'i} = delta_gg' delta_hh'   (P2)
    a, b, d, e, i = 1, 2, 2, 1, 2
    gs = [g for g in range(0, 6) if _tri(a, d, g)]
    hs = [h for h in range(0, 6) if _tri(b, e, h)]
    for g, h, gp, hp in itertools.product(gs, hs, gs, hs):
        if not (_tri(g, h, i) and _tri(gp, hp, i)):
            continue
        s = 0.0
        for c in range(0, 8):
            for f in range(0, 8):
                s += (c + 1) * (f + 1) * (g + 1) * (h + 1) * w9j(a, b, c, d, e, f, g, h, i) * w9j(a, b, c, d, e, f, gp, hp, i)
        assert abs(s - (1.0 if (g, h) == (gp, hp) else 0.0)) < 1e-12
    # F4 (the paper's W^(h): j = j' = S_target, k = 0):
    # W9j(j1,j2,J; k,k,0; j1',j2',J) = (-1)^(j1+j2'+J+k)/sqrt((2J+1)(2k+1)) {j1 j2 J; j2' j1' k}
    n = 0
    for j1, j2, J, k, j1p, j2p in itertools.product(range(0, 4), repeat=6):
        if _tri(j1, j2, J) and _tri(j1p, j2p, J) and _tri(j1, k, j1p) and _tri(j2, k, j2p):
            ref = (-1) ** ((j1 + j2p + J + k) // 2) / sqrt((J + 1) * (k + 1)) * w6j(j1, j2, J, j2p, j1p, k)
            assert abs(w9j(j1, j2, J, k, k, 0, j1p, j2p, J) - ref) < 1e-13
            n += 1
    assert n > 100
