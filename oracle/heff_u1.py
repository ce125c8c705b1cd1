"""ORACLE (test infrastructure only; never imported by the product path).

U(1)-only mode: H_eff * Psi for a problem whose sectors are labelled
by (N, 2 S_z) and whose coefficient per task is just the fermion sign times the two site elements -- the calculation
"just like for U(1) symmetry" that the SU(2) one is compared with.  Two things live here:

* heff_apply_u1: the plain definition, Eq. (2)/(3) with the three nested loops of
  PAPER.md:58-60 written out: F{p^F} += alpha_pos * A_pos{p^A} B{p^B} C{p^C} E{p^E} D_pos{p^D}^T with the Jordan-Wigner
  sign of SURVEY.md 8(c) C1.7.  A Psi sector is (il, b, 0, c, ir, 0), b / c in {0: |0>, 1: |up>, 2: |down>, 3: |up down>}.
* expand_problem: the SU(2) problem (reduced blocks) written out as a U(1) problem with Clebsch-Gordan coefficients
  (Wigner-Eckart; rows as in C2 / O5), either one U(1) sector per (SU(2) sector, M) or, merged, one
  per (N, 2 S_z) as a U(1) code would hold them; and the matching expansion / projection of Psi (O4 / O6).

Pins: tests/test_oracle_u1.py -- heff_apply_u1 on the expanded exact Hamiltonian reproduces the (N, S_z) spectrum of the
Jordan-Wigner Hamiltonian (oracle/fock.py, FCI); expand(SU(2) oracle result) = U(1) oracle result on the expansion;
merged = unmerged.
"""
import numpy as np

from gen.problem import OpFamily, Problem, Sector, SiteOp, Term

from .heff_dense import SITE_2S, SITE_N, SITE_STATES, _cg3, _full_keys, psi_sectors
from .wigner import cg

U1_SITE_N = (0, 1, 1, 2)
U1_SITE_M = (0, 1, -1, 0)
# oracle/heff_dense.SITE_STATES lists (multiplet, 2m) in the same order: |0>, |up>, |down>, |up down>
assert [(SITE_N[s], m) for s, m in SITE_STATES] == list(zip(U1_SITE_N, U1_SITE_M))


def psi_sectors_u1(problem):
    out = []
    for il, sl in enumerate(problem.sec_l):
        for b in range(4):
            for c in range(4):
                for ir, sr in enumerate(problem.sec_r):
                    if sl.N + U1_SITE_N[b] + U1_SITE_N[c] + sr.N != problem.n_tot:
                        continue
                    if sl.twoS + U1_SITE_M[b] + U1_SITE_M[c] + sr.twoS != problem.twoS_tot:
                        continue
                    out.append((il, b, 0, c, ir, 0))
    return out


def heff_apply_u1(problem, psi):
    """F = H_eff Psi, psi / F: {label: (D_l x D_r) array} over psi_sectors_u1 (absent = zero)."""
    assert problem.symmetry == "u1"
    labels = psi_sectors_u1(problem)
    have = set(labels)
    out = {lab: np.zeros((problem.sec_l[lab[0]].dim, problem.sec_r[lab[4]].dim)) for lab in labels}
    for t in problem.term:                                             # loop 1: operator-table rows
        fl = problem.fam_l[t.fam_l] if t.fam_l >= 0 else None
        fr = problem.fam_r[t.fam_r] if t.fam_r >= 0 else None
        oB, oC = problem.site[t.op_B], problem.site[t.op_C]
        dNr = 0 if fr is None else (-fr.dN if t.adj_r else fr.dN)
        pB, pC, pr = oB.dN & 1, oC.dN & 1, dNr & 1
        npos = problem.npos_of(t)
        alpha = np.ones(npos) if t.alpha is None else np.asarray(t.alpha, dtype=float)

        def transitions(fam, adj, secs):
            if fam is None:
                return [(i, i, -1) for i in range(len(secs))]
            return [((qo, qi, b) if adj else (qi, qo, b)) for b, (qo, qi) in enumerate(zip(fam.q_out, fam.q_in))]
        for li, lo, lb in transitions(fl, t.adj_l, problem.sec_l):     # loop 2: sector tasks of the row
            for ri, ro, rb in transitions(fr, t.adj_r, problem.sec_r):
                for bi in range(4):
                    for bo in range(4):
                        if oB.r[bo][bi] == 0.0:
                            continue
                        for ci in range(4):
                            for co in range(4):
                                if oC.r[co][ci] == 0.0:
                                    continue
                                src, dst = (li, bi, 0, ci, ri, 0), (lo, bo, 0, co, ro, 0)
                                if src not in psi or dst not in have:
                                    continue
                                nl = problem.sec_l[li].N
                                sgn = (-1) ** (pB * nl + pC * (nl + U1_SITE_N[bi]) + pr * (nl + U1_SITE_N[bi] + U1_SITE_N[ci]))
                                coef = sgn * oB.r[bo][bi] * oC.r[co][ci]
                                e = psi[src]
                                for pos in range(npos):                # loop 3: positions
                                    x = e
                                    if fl is not None:
                                        a = fl.data[lb][pos if fl.data[lb].shape[0] > 1 else 0]
                                        x = (a.T if t.adj_l else a) @ x
                                    if fr is not None:
                                        d = fr.data[rb][pos if fr.data[rb].shape[0] > 1 else 0]
                                        x = x @ (d if t.adj_r else d.T)
                                    out[dst] += coef * alpha[pos] * x
    return out


def flatten_u1(problem, red, labels=None):
    labels = psi_sectors_u1(problem) if labels is None else labels
    return np.concatenate([np.asarray(red[s]).ravel() if s in red else
                           np.zeros(problem.sec_l[s[0]].dim * problem.sec_r[s[4]].dim) for s in labels])


def unflatten_u1(problem, vec, labels=None):
    labels = psi_sectors_u1(problem) if labels is None else labels
    out, off = {}, 0
    for s in labels:
        m, n = problem.sec_l[s[0]].dim, problem.sec_r[s[4]].dim
        out[s] = np.asarray(vec[off:off + m * n]).reshape(m, n)
        off += m * n
    return out


# ----------------------------------------------------------------------------------------------------------------
# SU(2) problem -> U(1) problem
# ----------------------------------------------------------------------------------------------------------------
class U1Map:
    """Where the multiplet sector i of a block, at magnetic number M, sits in the U(1) sector table:
    pos[(i, M)] = (U(1) sector index, first row inside it)."""

    def __init__(self, secs, merged):
        self.sectors, self.pos = [], {}
        if not merged:
            for i, s in enumerate(secs):
                for m in range(-s.twoS, s.twoS + 1, 2):
                    self.pos[(i, m)] = (len(self.sectors), 0)
                    self.sectors.append(Sector(s.N, m, s.dim))
            return
        groups = {}
        for i, s in enumerate(secs):
            for m in range(-s.twoS, s.twoS + 1, 2):
                groups.setdefault((s.N, m), []).append(i)
        for (n, m), members in sorted(groups.items()):
            off = 0
            for i in members:
                self.pos[(i, m)] = (len(self.sectors), off)
                off += secs[i].dim
            self.sectors.append(Sector(n, m, off))


def expand_problem(problem, merged=False, with_data=True):
    """The SU(2) problem written out in the (N, 2 S_z) basis.  merged: one U(1) sector per (N, 2 S_z) (the multiplet
    sectors of equal N and admissible S stacked), as a U(1) calculation holds them -- the flavour whose CC the paper's
    R_CC compares with; otherwise one per (multiplet sector, M).  with_data=False: structure only
    (sector tables, block lists, rows), for counting.  Returns (u1_problem, (map_l, map_r))."""
    assert problem.symmetry == "su2"
    maps = (U1Map(problem.sec_l, merged), U1Map(problem.sec_r, merged))

    def expand_families(fams, secs, umap):
        out, index = [], {}
        for f, fam in enumerate(fams):
            for q in range(-fam.twoK, fam.twoK + 1, 2):
                blocks = {}
                for b, (qo, qi) in enumerate(zip(fam.q_out, fam.q_in)):
                    so, si = secs[qo].twoS, secs[qi].twoS
                    for mi in range(-si, si + 1, 2):
                        mo = mi + q
                        if abs(mo) > so:
                            continue
                        w = cg(fam.twoK, q, si, mi, so, mo)            # Wigner-Eckart, convention of C1.4
                        if w == 0.0:
                            continue
                        (uo, ro), (ui, ci) = umap.pos[(qo, mo)], umap.pos[(qi, mi)]
                        blocks.setdefault((uo, ui), []).append((ro, ci, w, b))
                keys = sorted(blocks)
                data = []
                for (uo, ui) in keys:
                    if not with_data:
                        data.append(None)
                        continue
                    arr = np.zeros((fam.npos, umap.sectors[uo].dim, umap.sectors[ui].dim))
                    for ro, ci, w, b in blocks[(uo, ui)]:
                        blk = fam.data[b]
                        arr[:, ro:ro + blk.shape[1], ci:ci + blk.shape[2]] += w * blk
                    data.append(arr)
                index[(f, q)] = len(out)
                out.append(OpFamily(dN=fam.dN, twoK=q, npos=fam.npos, q_out=[k[0] for k in keys], q_in=[k[1] for k in keys],
                                    data=data, name="%s[q=%d]" % (fam.name, q)))
        return out, index

    fam_l, idx_l = expand_families(problem.fam_l, problem.sec_l, maps[0])
    fam_r, idx_r = expand_families(problem.fam_r, problem.sec_r, maps[1])
    site, idx_s = [], {}
    for o, op in enumerate(problem.site):
        for q in range(-op.twoK, op.twoK + 1, 2):
            r = np.zeros((4, 4))
            for so, (sgo, mo) in enumerate(SITE_STATES):
                for si, (sgi, mi) in enumerate(SITE_STATES):
                    if op.r[sgo][sgi] != 0.0 and mo == mi + q:
                        r[so, si] = cg(op.twoK, q, SITE_2S[sgi], mi, SITE_2S[sgo], mo) * op.r[sgo][sgi]
            idx_s[(o, q)] = len(site)
            site.append(SiteOp(dN=op.dN, twoK=q, r=r, name="%s[q=%d]" % (op.name, q)))
    terms = []
    for t in problem.term:
        kl = problem.fam_l[t.fam_l].twoK if t.fam_l >= 0 else 0
        kr = problem.fam_r[t.fam_r].twoK if t.fam_r >= 0 else 0
        kB, kC = problem.site[t.op_B].twoK, problem.site[t.op_C].twoK
        k1, k2 = t.twoK_L, t.twoK_R
        npos = problem.npos_of(t)
        alpha = np.ones(npos) if t.alpha is None else np.asarray(t.alpha, dtype=float)
        for ql in range(-kl, kl + 1, 2):
            for qB in range(-kB, kB + 1, 2):
                for qC in range(-kC, kC + 1, 2):
                    qr = -(ql + qB + qC)
                    if abs(qr) > kr or (qr + kr) % 2:
                        continue
                    w = (cg(kl, ql, kB, qB, k1, ql + qB) * cg(kC, qC, kr, qr, k2, qC + qr)
                         * cg(k1, ql + qB, k2, qC + qr, 0, 0))
                    if w == 0.0:
                        continue
                    # adjoint tensor of a family: T~_q = (-1)^(k+q) (T_-q)^dagger (C1.3): component -q read transposed
                    fl = fr = -1
                    if t.fam_l >= 0:
                        fl = idx_l[(t.fam_l, -ql if t.adj_l else ql)]
                        if t.adj_l:
                            w *= (-1) ** ((kl + ql) // 2)
                    if t.fam_r >= 0:
                        fr = idx_r[(t.fam_r, -qr if t.adj_r else qr)]
                        if t.adj_r:
                            w *= (-1) ** ((kr + qr) // 2)
                    terms.append(Term(fam_l=fl, fam_r=fr, op_B=idx_s[(t.op_B, qB)], op_C=idx_s[(t.op_C, qC)], twoK_L=0,
                                      twoK_R=0, alpha=w * alpha, adj_l=t.adj_l if fl >= 0 else 0,
                                      adj_r=t.adj_r if fr >= 0 else 0, name="%s[%d,%d,%d,%d]" % (t.name, ql, qB, qC, qr)))
    u1 = Problem(n_tot=problem.n_tot, twoS_tot=problem.twoS_tot, sec_l=maps[0].sectors, sec_r=maps[1].sectors,
                 fam_l=fam_l, fam_r=fam_r, site=site, term=terms, meta=dict(problem.meta, u1_merged=merged), symmetry="u1")
    return u1, maps


def expand_psi_u1(problem, u1, maps, psi_red):
    """O4: Psi in the (N, 2 S_z) basis at M_tot = S_tot from the reduced blocks."""
    out = {lab: np.zeros((u1.sec_l[lab[0]].dim, u1.sec_r[lab[4]].dim)) for lab in psi_sectors_u1(u1)}
    for label, blk in psi_red.items():
        il, _, _, _, ir, _ = label
        for ml, b, c, mr, mb, mc in _full_keys(problem, label):
            w = _cg3(problem, label, ml, mb, mc, mr)
            if w == 0.0:
                continue
            (ul, r0), (ur, c0) = maps[0].pos[(il, ml)], maps[1].pos[(ir, mr)]
            out[(ul, b, 0, c, ur, 0)][r0:r0 + blk.shape[0], c0:c0 + blk.shape[1]] += w * blk
    return out


def project_psi_u1(problem, maps, f_u1):
    """O6: back onto the coupled basis."""
    red = {}
    for label in psi_sectors(problem):
        il, _, _, _, ir, _ = label
        dl, dr = problem.sec_l[il].dim, problem.sec_r[ir].dim
        acc = np.zeros((dl, dr))
        for ml, b, c, mr, mb, mc in _full_keys(problem, label):
            w = _cg3(problem, label, ml, mb, mc, mr)
            if w == 0.0:
                continue
            (ul, r0), (ur, c0) = maps[0].pos[(il, ml)], maps[1].pos[(ir, mr)]
            acc += w * f_u1[(ul, b, 0, c, ur, 0)][r0:r0 + dl, c0:c0 + dr]
        red[label] = acc
    return red
