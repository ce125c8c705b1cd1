"""Seeded synthetic workloads with the shapes of the paper's.

The paper measures on F2 CAS(18,18), N2 CAS(14,28) and FeMoco CAS(54,54)/(113,76) with
D = 512...24576; those integrals and matrix-product states are not
available, so the BASELINE.json configs stand in for them: half filling, singlet target,
middle bond, N^2 position batches, block sectors (N,S) with multiplicities up to ~550.

Input generation only: sector tables, random reduced operator blocks with the correct
selection rules, operator-table rows, integrals, Psi.  The method's arithmetic (recoupling
coefficients, task enumeration, products) is NOT here.
"""
from math import comb, exp, sqrt

import numpy as np

from . import rng
from .problem import OpFamily, Problem, Sector, SiteOp, Term

CONFIGS = {
    # name: L (orbitals), N (electrons), twoS, D (multiplets kept), xi (integral decay length)
    "cfg1": dict(L=6, N=6, twoS=0, D=16, xi=2.0),
    "cfg2": dict(L=20, N=20, twoS=0, D=256, xi=2.0),
    "cfg3": dict(L=40, N=40, twoS=0, D=1024, xi=2.0),
    "cfg4": dict(L=76, N=76, twoS=0, D=4096, xi=6.0),
    # small stand-ins of the same family for fast tests
    "mini": dict(L=8, N=8, twoS=0, D=24, xi=2.0),
    "midi": dict(L=12, N=12, twoS=0, D=64, xi=2.0),
    # profiling stand-in for cfg4: the same sector tables and block sizes (69-547), but every operator
    # family keeps only its first 24 positions, so that one apply takes ~1 s and fits an ncu replay
    "cfg4p": dict(L=76, N=76, twoS=0, D=4096, xi=6.0, pos_cap=24),
}

TAG_T, TAG_V, TAG_PSI, TAG_ALPHA, TAG_OP = 1, 2, 3, 4, 16


# ----------------------------------------------------------------------------- integrals
def integrals(L, seed=0, xi=2.0):
    """t_ij symmetric, sigma = 0.1 exp(-|i-j|/xi); (ij|kl) 8-fold symmetric,
    sigma = 0.1 exp(-(|i-j|+|k-l|)/xi); each value drawn once from the canonical (sorted)
    representative of its symmetry orbit (reading G11 of BASELINE.json configs[0])."""
    t = np.zeros((L, L))
    for i in range(L):
        for j in range(L):
            a, b = min(i, j), max(i, j)
            t[i, j] = 0.1 * exp(-abs(i - j) / xi) * float(rng.normal(seed, TAG_T, a * L + b))
    v = np.zeros((L, L, L, L))
    for i in range(L):
        for j in range(L):
            for k in range(L):
                for l in range(L):
                    p, q = (min(i, j), max(i, j)), (min(k, l), max(k, l))
                    if q < p:
                        p, q = q, p
                    idx = ((p[0] * L + p[1]) * L + q[0]) * L + q[1]
                    v[i, j, k, l] = 0.1 * exp(-(abs(i - j) + abs(k - l)) / xi) * float(rng.normal(seed, TAG_V, idx))
    return t, v


# ----------------------------------------------------------------------------- sectors
def weyl_paldus(n, N, twoS):
    """Number of spin-S multiplets of N electrons in n orbitals."""
    if N < 0 or N > 2 * n or twoS < 0 or (N - twoS) % 2 or twoS > min(N, 2 * n - N):
        return 0
    a = (N - twoS) // 2
    b = (N + twoS) // 2 + 1
    return (twoS + 1) * comb(n + 1, a) * comb(n + 1, b) // (n + 1)


def block_sectors(n_block, L, N, twoS_tot, D):
    """Sector table of a block of n_block orbitals keeping D multiplets (reading G12):
    weights W(n_block,N_b,S_b) * W(L-n_block, N-N_b, S_b) inside the window
    |N_b - n_block N/L| <= 2, S_b <= 2; largest-remainder rounding, capped at the number of
    multiplets that exist.  If all multiplets of the block fit in D, the block is complete."""
    assert twoS_tot == 0
    total = sum(weyl_paldus(n_block, nb, s) for nb in range(2 * n_block + 1) for s in range(nb % 2, nb + 1, 2))
    cand = []
    for nb in range(2 * n_block + 1):
        for s in range(nb % 2, min(nb, 2 * n_block - nb) + 1, 2):
            cap = weyl_paldus(n_block, nb, s)
            if cap == 0:
                continue
            if total <= D:
                cand.append((nb, s, cap, float(cap)))
                continue
            if abs(nb - n_block * N / L) > 2 or s > 4:
                continue
            w = cap * weyl_paldus(L - n_block, N - nb, s)
            if w > 0:
                cand.append((nb, s, cap, float(w)))
    if total <= D:
        return [Sector(nb, s, cap) for nb, s, cap, _ in cand]
    wsum = sum(c[3] for c in cand)
    quota = [D * c[3] / wsum for c in cand]
    dims = [min(c[2], int(q)) for c, q in zip(cand, quota)]
    while sum(dims) < D:
        order = sorted((i for i in range(len(cand)) if dims[i] < cand[i][2]),
                       key=lambda i: (-(quota[i] - dims[i]), i))
        if not order:
            break
        for i in order[:D - sum(dims)]:
            dims[i] += 1
    return [Sector(c[0], c[1], d) for c, d in zip(cand, dims) if d > 0]


# ----------------------------------------------------------------------------- site operators
_S2, _S32 = sqrt(2.0), sqrt(1.5)


def site_table():
    """The site operators (reduced elements in Wigner-Eckart convention B, SURVEY.md 8(c)
    C1.6; every entry is re-derived by brute force in tests/test_oracle_fock.py) and, for
    Hermitian-conjugate rows, adj[name] = (name of the adjoint tensor's operator, factor):
    adjoint-tensor(O) = factor * O_adj."""
    def op(name, dN, twoK, entries):
        r = np.zeros((3, 3))
        for (o, i), val in entries.items():
            r[o, i] = val
        return SiteOp(dN=dN, twoK=twoK, r=r, name=name)

    ops = [
        op("1", 0, 0, {(0, 0): 1.0, (1, 1): 1.0, (2, 2): 1.0}),
        op("c+", +1, 1, {(1, 0): 1.0, (2, 1): _S2}),
        op("c~", -1, 1, {(0, 1): -_S2, (1, 2): 1.0}),
        op("A0", +2, 0, {(2, 0): _S2}),
        op("A~0", -2, 0, {(0, 2): -_S2}),
        op("B0", 0, 0, {(1, 1): 1.0 / _S2, (2, 2): _S2}),
        op("B1", 0, 2, {(1, 1): -_S32}),
        op("D", 0, 0, {(2, 2): 1.0}),                     # double-occupancy projector n_u n_d
    ]
    adj = {"1": ("1", 1.0), "c+": ("c~", 1.0), "c~": ("c+", -1.0), "A0": ("A~0", -1.0), "A~0": ("A0", -1.0),
           "B0": ("B0", 1.0), "B1": ("B1", -1.0), "D": ("D", 1.0)}
    return ops, adj


# ----------------------------------------------------------------------------- operator families
def _family_blocks(sec, dN, twoK):
    """All (q_out, q_in) sector pairs allowed by particle number and the triangle rule."""
    out = []
    for io, so in enumerate(sec):
        for ii, si in enumerate(sec):
            if so.N == si.N + dN and abs(si.twoS - twoK) <= so.twoS <= si.twoS + twoK and (si.twoS + twoK + so.twoS) % 2 == 0:
                out.append((io, ii))
    return out


def make_family(sec, dN, twoK, npos, seed, tag, name, symmetric=False, fill=True):
    """Random family: every stored entry N(0, 1/sqrt(dim_in)) so that |A E D^T| stays O(1)."""
    blocks = _family_blocks(sec, dN, twoK)
    data = []
    for b, (io, ii) in enumerate(blocks):
        m, k = sec[io].dim, sec[ii].dim
        if fill:
            arr = rng.normal_array(seed, tag * 4096 + b, (npos, m, k)) / sqrt(k)
            if symmetric and io == ii:
                arr = 0.5 * (arr + np.swapaxes(arr, 1, 2))
        else:
            arr = None
        data.append(arr)
    fam = OpFamily(dN=dN, twoK=twoK, npos=npos, q_out=[b[0] for b in blocks], q_in=[b[1] for b in blocks],
                   data=data, name=name)
    return fam


def synthetic_problem(L, N, twoS, D, xi=2.0, seed=0, fill=True, site_terms=True, hermitian=True, pos_cap=None):
    """Random-operator problem at the middle bond with the row classes of SURVEY.md 8(c) C3:
    local, 1+3, 2+2 pair (A^S P~^S), 2+2 particle-hole (B^S Q^S), plus a few site-involving
    rows; every non-self-adjoint row is accompanied by its Hermitian conjugate (adjoint
    flags on the same stored families) when `hermitian`."""
    nl = L // 2 - 1
    nr = L - nl - 2
    sec_l = block_sectors(nl, L, N, twoS, D)
    sec_r = block_sectors(nr, L, N, twoS, D)
    site, site_adj = site_table()
    sid = {o.name: i for i, o in enumerate(site)}
    pairs_le = [(i, j) for i in range(nl) for j in range(i, nl)]
    pairs_lt = [(i, j) for i in range(nl) for j in range(i + 1, nl)]
    if pos_cap is not None:
        pairs_le, pairs_lt = pairs_le[:pos_cap], pairs_lt[:pos_cap]

    fam_l, fam_r, terms = [], [], []

    def add(side, dN, twoK, npos, name, symmetric=False):
        fams, sec = (fam_l, sec_l) if side == "l" else (fam_r, sec_r)
        tag = TAG_OP + len(fam_l) * 2 if side == "l" else TAG_OP + len(fam_r) * 2 + 1
        fams.append(make_family(sec, dN, twoK, npos, seed, tag, name, symmetric=symmetric, fill=fill))
        return len(fams) - 1

    def alpha_for(tag, pos_dist):
        """integral-like alpha per position: N(0, 0.1 exp(-dist/xi))."""
        d = np.asarray(pos_dist, dtype=float)
        z = rng.normal(seed, TAG_ALPHA * 4096 + tag, np.arange(len(d)))
        return 0.1 * np.exp(-d / xi) * z

    def add_term(fl, fr, oB, oC, k1, alpha, name, self_adjoint=False):
        terms.append(Term(fam_l=fl, fam_r=fr, op_B=sid[oB], op_C=sid[oC], twoK_L=k1, twoK_R=k1,
                          alpha=None if alpha is None else np.array(alpha, dtype=float), name=name))
        if self_adjoint or not hermitian:
            return
        # X^dagger = s_lB s_Cr s_12 [[O~_l x O~_B]^k1 x [O~_C x O~_r]^k1]^0 with s_XY = (-1)^(p_X p_Y)
        pl = fam_l[fl].parity if fl >= 0 else 0
        pr = fam_r[fr].parity if fr >= 0 else 0
        pB, pC = site[sid[oB]].parity, site[sid[oC]].parity
        sgn = (-1.0) ** (pl * pB + pC * pr + (pl + pB) * (pC + pr))
        (aB, fB), (aC, fC) = site_adj[oB], site_adj[oC]
        a = np.ones(1 if alpha is None else len(alpha)) if alpha is None else np.array(alpha, dtype=float)
        if alpha is None:
            npos = max(fam_l[fl].npos if fl >= 0 else 1, fam_r[fr].npos if fr >= 0 else 1)
            a = np.ones(npos)
        terms.append(Term(fam_l=fl, fam_r=fr, op_B=sid[aB], op_C=sid[aC], twoK_L=k1, twoK_R=k1,
                          alpha=a * (sgn * fB * fC), adj_l=1 if fl >= 0 else 0, adj_r=1 if fr >= 0 else 0,
                          name=name + "^H"))

    # local rows
    hl = add("l", 0, 0, 1, "H_l", symmetric=True)
    hr = add("r", 0, 0, 1, "H_r", symmetric=True)
    add_term(hl, -1, "1", "1", 0, None, "H_l", self_adjoint=True)
    add_term(-1, hr, "1", "1", 0, None, "H_r", self_adjoint=True)
    add_term(-1, -1, "B0", "1", 0, [0.3], "H_B:n", self_adjoint=True)
    add_term(-1, -1, "D", "1", 0, [0.7], "H_B:U", self_adjoint=True)
    add_term(-1, -1, "1", "B0", 0, [-0.2], "H_C:n", self_adjoint=True)
    add_term(-1, -1, "1", "D", 0, [0.6], "H_C:U", self_adjoint=True)

    # 1+3: c+_i(l) R~_i(r) and R_y(l) c~_y(r)
    cl = add("l", +1, 1, nl, "c+(l)")
    rr = add("r", -1, 1, nl, "R~(r)")
    add_term(cl, rr, "1", "1", 1, np.ones(nl), "c+R~")
    rl = add("l", +1, 1, nr, "R(l)")
    cr = add("r", -1, 1, nr, "c~(r)")
    add_term(rl, cr, "1", "1", 1, np.ones(nr), "Rc~")

    # 2+2 pair: A^S_ij(l) P~^S_ij(r), S=0 (i<=j), S=1 (i<j)
    a0 = add("l", +2, 0, len(pairs_le), "A0(l)")
    p0 = add("r", -2, 0, len(pairs_le), "P~0(r)")
    add_term(a0, p0, "1", "1", 0, alpha_for(1, [j - i for i, j in pairs_le]) * 10, "A0P0")
    if pairs_lt:
        a1 = add("l", +2, 2, len(pairs_lt), "A1(l)")
        p1 = add("r", -2, 2, len(pairs_lt), "P~1(r)")
        add_term(a1, p1, "1", "1", 2, alpha_for(2, [j - i for i, j in pairs_lt]) * 10, "A1P1")

    # 2+2 particle-hole: B^S_ij(l) Q^S_ij(r), i<=j (B_ji from the adjoint)
    b0 = add("l", 0, 0, len(pairs_le), "B0(l)")
    q0 = add("r", 0, 0, len(pairs_le), "Q0(r)")
    add_term(b0, q0, "1", "1", 0, alpha_for(3, [j - i for i, j in pairs_le]) * 10, "B0Q0")
    b1 = add("l", 0, 2, len(pairs_le), "B1(l)")
    q1 = add("r", 0, 2, len(pairs_le), "Q1(r)")
    add_term(b1, q1, "1", "1", 2, alpha_for(4, [j - i for i, j in pairs_le]) * 10, "B1Q1")

    if site_terms:
        # one-body hops and density couplings that involve the sites
        add_term(cl, -1, "c~", "1", 0, alpha_for(5, [nl - i for i in range(nl)]) * 10, "hop lB")
        add_term(cl, -1, "1", "c~", 1, alpha_for(6, [nl + 1 - i for i in range(nl)]) * 10, "hop lC")
        add_term(-1, cr, "c+", "1", 1, alpha_for(7, [y + 2 for y in range(nr)]) * 10, "hop Br")
        add_term(-1, cr, "1", "c+", 0, alpha_for(8, [y + 1 for y in range(nr)]) * 10, "hop Cr")
        add_term(-1, -1, "c+", "c~", 1, [0.25], "hop BC")
        add_term(-1, -1, "B0", "B0", 0, [0.4], "nn BC", self_adjoint=True)
        add_term(-1, -1, "B1", "B1", 2, [-0.35], "ss BC", self_adjoint=True)
        add_term(-1, -1, "A0", "A~0", 0, [0.15], "pair BC")
        add_term(b0, -1, "B0", "1", 0, alpha_for(9, [nl - i for i, j in pairs_le]) * 10, "B0(l) n_B")
        add_term(b1, -1, "B1", "1", 0, alpha_for(10, [nl - i for i, j in pairs_le]) * 10, "B1(l) s_B")
        add_term(b1, -1, "1", "B1", 2, alpha_for(11, [nl - i for i, j in pairs_le]) * 10, "B1(l) s_C")
        add_term(-1, q1, "B1", "1", 2, alpha_for(12, [j for i, j in pairs_le]) * 10, "s_B Q1(r)")
        add_term(a0, -1, "1", "A~0", 0, alpha_for(13, [nl - i for i, j in pairs_le]) * 10, "A0(l) A~0_C")
        add_term(cl, cr, "c+", "c~", 2, None, "c+ c+_B c~_C c~ (k1=1)")
        add_term(cl, rr, "B1", "1", 1, np.ones(nl) * 0.5, "c+ s_B R~")

    prob = Problem(n_tot=N, twoS_tot=twoS, sec_l=sec_l, sec_r=sec_r, fam_l=fam_l, fam_r=fam_r, site=site,
                   term=terms, meta=dict(L=L, N=N, D=D, xi=xi, seed=seed, nl=nl, nr=nr))
    return prob


def config_problem(name, seed=0, fill=True):
    c = CONFIGS[name]
    return synthetic_problem(c["L"], c["N"], c["twoS"], c["D"], xi=c["xi"], seed=seed, fill=fill, pos_cap=c.get("pos_cap"))


def random_psi(psi_len, seed=0):
    """Psi: N(0,1) per element, normalised in the Frobenius norm of the reduced blocks."""
    x = rng.normal_array(seed, TAG_PSI, (psi_len,))
    return x / np.linalg.norm(x)
