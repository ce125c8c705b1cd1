"""ORACLE (test infrastructure only; never imported by the product path).

H_eff * Psi by its plain definition.

The SU(2) method "can be performed just like for U(1) symmetry except that ... each result is
multiplied with an additional scalar".  So the oracle does the U(1)
computation: it expands every reduced (Wigner-Eckart) block operator and the reduced wave
function to the M-resolved basis with Clebsch-Gordan coefficients, applies the four-subsystem
product of PAPER.md Eq. (2)/(3) component by component with the Jordan-Wigner
signs, and projects back onto the coupled basis.  No 6j/9j symbol is used anywhere here; the
recoupling coefficients of the fast path must reproduce this result.

Coupling tree ((l,B)J1,(C,r)J2)S_tot (the tree of the paper's W^(l), W^(r), W^(h) tables,
PAPER.md:92-106).  A Psi sector label is (il, sB, twoJ1, sC, ir, twoJ2): il/ir index
problem.sec_l/sec_r, sB/sC in {0,1,2} are the site multiplets (N=0,S=0), (1,1/2), (2,0).

Pins: tests/test_oracle_heff.py (P5, P8, P9, P10 of SURVEY.md 8(c) C6).
"""
import numpy as np

from .wigner import cg

SITE_N = (0, 1, 2)            # particle number of site multiplet sigma
SITE_2S = (0, 1, 0)           # doubled spin of site multiplet sigma
# M-resolved site states: (sigma, two_m)
SITE_STATES = ((0, 0), (1, 1), (1, -1), (2, 0))


def _triangle(a, b, c):
    return (a + b + c) % 2 == 0 and abs(a - b) <= c <= a + b


def psi_sectors(problem):
    """All Psi sector labels s = (il, sB, twoJ1, sC, ir, twoJ2) allowed by particle number
    and the triangle rules of the coupling tree (SURVEY.md section 8 notation)."""
    out = []
    for il, sl in enumerate(problem.sec_l):
        for sB in range(3):
            for sC in range(3):
                for ir, sr in enumerate(problem.sec_r):
                    if sl.N + SITE_N[sB] + SITE_N[sC] + sr.N != problem.n_tot:
                        continue
                    for j1 in range(abs(sl.twoS - SITE_2S[sB]), sl.twoS + SITE_2S[sB] + 1, 2):
                        for j2 in range(abs(sr.twoS - SITE_2S[sC]), sr.twoS + SITE_2S[sC] + 1, 2):
                            if _triangle(j1, j2, problem.twoS_tot):
                                out.append((il, sB, j1, sC, ir, j2))
    return out


def _cg3(problem, label, ml, mb, mc, mr):
    """<S_l M_l; s_B m_B|J1 M1> <s_C m_C; S_r M_r|J2 M2> <J1 M1; J2 M2|S_tot S_tot>  (O4)."""
    il, sB, j1, sC, ir, j2 = label
    sl, sr = problem.sec_l[il].twoS, problem.sec_r[ir].twoS
    m1, m2 = ml + mb, mc + mr
    return (cg(sl, ml, SITE_2S[sB], mb, j1, m1) * cg(SITE_2S[sC], mc, sr, mr, j2, m2)
            * cg(j1, m1, j2, m2, problem.twoS_tot, problem.twoS_tot))


def _full_keys(problem, label):
    """M-resolved components (ml, b, c, mr) reachable from one reduced sector at M_tot = S_tot."""
    il, sB, j1, sC, ir, j2 = label
    sl, sr = problem.sec_l[il].twoS, problem.sec_r[ir].twoS
    for b, (sgb, mb) in enumerate(SITE_STATES):
        if sgb != sB:
            continue
        for c, (sgc, mc) in enumerate(SITE_STATES):
            if sgc != sC:
                continue
            for ml in range(-sl, sl + 1, 2):
                mr = problem.twoS_tot - ml - mb - mc
                if abs(mr) > sr or (mr + sr) % 2:
                    continue
                yield ml, b, c, mr, mb, mc


def expand_psi(problem, psi_red):
    """O4: Psi_full[(il, M_l, b, c, ir, M_r)] = sum_{J1,J2} CG CG CG * Psi_red[s]."""
    full = {}
    for label, blk in psi_red.items():
        il, sB, j1, sC, ir, j2 = label
        for ml, b, c, mr, mb, mc in _full_keys(problem, label):
            w = _cg3(problem, label, ml, mb, mc, mr)
            if w == 0.0:
                continue
            key = (il, ml, b, c, ir, mr)
            if key in full:
                full[key] = full[key] + w * blk
            else:
                full[key] = w * blk
    return full


def project_psi(problem, full, labels):
    """O6: F_red[s] = sum over M-components of CG CG CG * F_full."""
    red = {}
    for label in labels:
        il, sB, j1, sC, ir, j2 = label
        acc = 0.0
        for ml, b, c, mr, mb, mc in _full_keys(problem, label):
            key = (il, ml, b, c, ir, mr)
            if key in full:
                acc = acc + _cg3(problem, label, ml, mb, mc, mr) * full[key]
        if isinstance(acc, float):
            acc = np.zeros((problem.sec_l[il].dim, problem.sec_r[ir].dim))
        red[label] = acc
    return red


def _block_transitions(fam, adj, sectors):
    """For a block operator family (or identity: fam None): list of
    (i_in, i_out, blockindex, transposed) of the operator actually applied."""
    if fam is None:
        return [(i, i, -1, False) for i in range(len(sectors))]
    if not adj:
        return [(qi, qo, b, False) for b, (qo, qi) in enumerate(zip(fam.q_out, fam.q_in))]
    return [(qo, qi, b, True) for b, (qo, qi) in enumerate(zip(fam.q_out, fam.q_in))]


def _block_element_factor(two_k, q, adj, s_in, m_in, s_out, m_out):
    """Scalar multiplying the reduced block for the component q of the applied operator,
    ket (s_in, m_in) -> bra (s_out, m_out).  Wigner-Eckart (C1.4) for the family itself;
    for its adjoint tensor T~_q = (-1)^(k+q) (T_{-q})^dagger (C1.3) the element is
    (-1)^(k+q) <S_in M_in|T_{-q}|S_out M_out>."""
    if not adj:
        return cg(two_k, q, s_in, m_in, s_out, m_out)
    return (-1) ** ((two_k + q) // 2) * cg(two_k, -q, s_out, m_out, s_in, m_in)


def apply_full(problem, psi_full, terms=None):
    """O5: F_full = sum_rows X_row Psi_full, each row applied component by component."""
    out = {}
    term_list = problem.term if terms is None else terms
    for t in term_list:
        fl = problem.fam_l[t.fam_l] if t.fam_l >= 0 else None
        fr = problem.fam_r[t.fam_r] if t.fam_r >= 0 else None
        oB, oC = problem.site[t.op_B], problem.site[t.op_C]
        kl = fl.twoK if fl is not None else 0
        kr = fr.twoK if fr is not None else 0
        kB, kC = oB.twoK, oC.twoK
        k1, k2 = t.twoK_L, t.twoK_R
        dNl = 0 if fl is None else (-fl.dN if t.adj_l else fl.dN)
        dNr = 0 if fr is None else (-fr.dN if t.adj_r else fr.dN)
        pB, pC, pr = oB.dN & 1, oC.dN & 1, dNr & 1
        npos = problem.npos_of(t)
        alpha = np.ones(npos) if t.alpha is None else np.asarray(t.alpha, dtype=float)
        ltrans = _block_transitions(fl, t.adj_l, problem.sec_l)
        rtrans = _block_transitions(fr, t.adj_r, problem.sec_r)
        for ql in range(-kl, kl + 1, 2):
            for qB in range(-kB, kB + 1, 2):
                for qC in range(-kC, kC + 1, 2):
                    qr = -(ql + qB + qC)
                    if abs(qr) > kr or (qr + kr) % 2:
                        continue
                    w_op = (cg(kl, ql, kB, qB, k1, ql + qB) * cg(kC, qC, kr, qr, k2, qC + qr)
                            * cg(k1, ql + qB, k2, qC + qr, 0, 0))
                    if w_op == 0.0:
                        continue
                    for key, blk in psi_full.items():
                        il_in, ml_in, b_in, c_in, ir_in, mr_in = key
                        sgb_in, mb_in = SITE_STATES[b_in]
                        sgc_in, mc_in = SITE_STATES[c_in]
                        # site B element <sigma m|O_B,q|sigma' m'> = <k q; s' m'|s m> r[sigma,sigma']
                        sgb = sgb_in + oB.dN
                        sgc = sgc_in + oC.dN
                        if not (0 <= sgb <= 2 and 0 <= sgc <= 2):
                            continue
                        mb, mc = mb_in + qB, mc_in + qC
                        eB = cg(kB, qB, SITE_2S[sgb_in], mb_in, SITE_2S[sgb], mb) * oB.r[sgb][sgb_in]
                        eC = cg(kC, qC, SITE_2S[sgc_in], mc_in, SITE_2S[sgc], mc) * oC.r[sgc][sgc_in]
                        if eB == 0.0 or eC == 0.0:
                            continue
                        b_out = SITE_STATES.index((sgb, mb))
                        c_out = SITE_STATES.index((sgc, mc))
                        n_l_in = problem.sec_l[il_in].N
                        # fermion sign with KET particle numbers (C1.7)
                        sgn = (-1) ** (pB * n_l_in + pC * (n_l_in + SITE_N[sgb_in])
                                       + pr * (n_l_in + SITE_N[sgb_in] + SITE_N[sgc_in]))
                        for (li, lo, lb, ltr) in ltrans:
                            if li != il_in:
                                continue
                            s_li, s_lo = problem.sec_l[li].twoS, problem.sec_l[lo].twoS
                            ml = ml_in + ql
                            if abs(ml) > s_lo:
                                continue
                            el = 1.0 if fl is None else _block_element_factor(kl, ql, t.adj_l, s_li, ml_in, s_lo, ml)
                            if el == 0.0:
                                continue
                            for (ri, ro, rb, rtr) in rtrans:
                                if ri != ir_in:
                                    continue
                                s_ri, s_ro = problem.sec_r[ri].twoS, problem.sec_r[ro].twoS
                                mr = mr_in + qr
                                if abs(mr) > s_ro:
                                    continue
                                er = 1.0 if fr is None else _block_element_factor(kr, qr, t.adj_r, s_ri, mr_in, s_ro, mr)
                                if er == 0.0:
                                    continue
                                coef = w_op * eB * eC * sgn * el * er
                                contrib = _sum_over_positions(fl, lb, ltr, fr, rb, rtr, alpha, blk)
                                okey = (lo, ml, b_out, c_out, ro, mr)
                                if okey in out:
                                    out[okey] += coef * contrib
                                else:
                                    out[okey] = coef * contrib
    return out


def _sum_over_positions(fl, lb, ltr, fr, rb, rtr, alpha, e):
    """sum_pos alpha_pos * A_pos E D_pos^T, written out as the paper's innermost loop over the
    position index ("three nested loops", the third over the positions); A, D = the
    applied l / r operator blocks (transposed if adjoint).  A family with a single position (or the
    identity: family None) contributes the same block at every pos.  Nothing is folded, factored
    or reordered here: one term alpha_pos * (A_pos @ E) @ D_pos^T per position, added in index order.
    E may carry leading batch axes (..., k, n)."""
    acc = 0.0
    for pos in range(len(alpha)):
        x = e
        if fl is not None:
            a = fl.data[lb][pos if fl.data[lb].shape[0] > 1 else 0]
            x = np.matmul(a.T if ltr else a, x)
        if fr is not None:
            d = fr.data[rb][pos if fr.data[rb].shape[0] > 1 else 0]
            x = np.matmul(x, d if rtr else d.T)
        acc = acc + alpha[pos] * x
    return acc


def heff_apply(problem, psi_red, check_leak=True, terms=None):
    """F_red = H_eff Psi_red (O1-O6).  psi_red: {label: (D_l x D_r) array}; sectors absent
    from psi_red are zero.  Returns {label: array} over ALL sectors of psi_sectors()."""
    labels = psi_sectors(problem)
    full = expand_psi(problem, psi_red)
    f_full = apply_full(problem, full, terms=terms)
    f_red = project_psi(problem, f_full, labels)
    if check_leak:
        back = expand_psi(problem, f_red)
        num, den = 0.0, 0.0
        for key in set(back) | set(f_full):
            x = f_full.get(key)
            y = back.get(key)
            if x is None:
                x = np.zeros_like(y)
            if y is None:
                y = np.zeros_like(x)
            num += float(((x - y) ** 2).sum())
            den += float((x ** 2).sum())
        if num > 1e-22 * max(den, 1e-300) and num > 1e-26:
            raise ValueError("operator table is not a scalar: leakage %.3e of %.3e" % (num ** 0.5, den ** 0.5))
    return f_red


def flatten(problem, red, labels=None):
    labels = psi_sectors(problem) if labels is None else labels
    return np.concatenate([red[s].ravel() if s in red else
                           np.zeros(problem.sec_l[s[0]].dim * problem.sec_r[s[4]].dim) for s in labels])


def unflatten(problem, vec, labels=None):
    labels = psi_sectors(problem) if labels is None else labels
    out, off = {}, 0
    for s in labels:
        m, n = problem.sec_l[s[0]].dim, problem.sec_r[s[4]].dim
        out[s] = np.asarray(vec[off:off + m * n]).reshape(m, n)
        off += m * n
    return out


def heff_matrix(problem):
    """Dense matrix of H_eff in the reduced basis (tiny problems only): for every input
    sector the batch of all its unit vectors is pushed through heff_apply at once."""
    labels = psi_sectors(problem)
    dims = [problem.sec_l[s[0]].dim * problem.sec_r[s[4]].dim for s in labels]
    offs = np.concatenate([[0], np.cumsum(dims)])
    h = np.zeros((offs[-1], offs[-1]))
    for si, s in enumerate(labels):
        m, n = problem.sec_l[s[0]].dim, problem.sec_r[s[4]].dim
        f = heff_apply(problem, {s: np.eye(m * n).reshape(m * n, m, n)}, check_leak=False)
        for so, lab in enumerate(labels):
            blk = f[lab]
            if blk.ndim == 3:
                h[offs[so]:offs[so + 1], offs[si]:offs[si + 1]] = blk.reshape(m * n, -1).T
    return h
