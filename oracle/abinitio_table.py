"""ORACLE-SIDE generator (test infrastructure only; never imported by the product path).

Builds the EXACT operator-table / sector-tables of the ab initio Hamiltonian
H = sum t_ij E_ij + 1/2 sum (ij|kl) X(i,k,l,j)  (Eq. (1), spin-free reading G7) for
a two-site superblock l | B | C | r of a SMALL orbital chain, with normal and pre-contracted
("complementary") block operators in reduced (Wigner-Eckart) form.

The paper prints no operator table ("paper is silent").  This module derives
it mechanically instead of from hand-derived identities:

 1. every elementary string  c+_is c_js  /  c+_is c+_kt c_lt c_js  is written as
    sum_q I[q1..qn] T1_q1 ... Tn_qn with T = c+ or c~ (C1.3) and I the spin-invariant tensor;
 2. the operators are stably sorted by subsystem (l,B,C,r) with the fermionic permutation
    sign (operators on different subsystems anticommute; the order inside a subsystem is kept);
 3. I is expanded in the orthonormal coupling schemes
       [[O_l x O_B]^k1 x [O_C x O_r]^k1]^0,  O_X = coupled product of the operators on X,
    (alpha_scheme = <W_scheme | I>, completeness checked);
 4. rows that differ only in the operator of one block are summed over that block's orbital
    indices: the pre-contraction N^4 -> N^2 of PAPER.md:43;
 5. block operators are built in the block's own Fock space and reduced in its multiplet basis.

The result is pinned end to end (P9): the spectrum of H_eff equals the spectrum of the
Jordan-Wigner Hamiltonian in the (N, S) sector when the blocks are untruncated.
"""
import itertools

import numpy as np

from gen.problem import OpFamily, Problem, Sector, SiteOp, Term
from .fock import FockSpace, TensorOp, couple
from .multiplets import full_multiplet_basis, reduce_tensor, site_multiplet_basis, truncate_basis
from .wigner import cg

_HALF = (1, -1)     # doubled projections of a rank-1/2 tensor


def _invariant_one_body():
    """E_ij = sum_s c+_is c_js = sum_q I[q1,q2] (c+_i)_q1 (c~_j)_q2 with c_u = c~_{-1/2},
    c_d = -c~_{+1/2}  (C1.3)."""
    return {(+1, -1): 1.0, (-1, +1): -1.0}


def _invariant_two_body():
    """X(i,k,l,j) = sum_st c+_is c+_kt c_lt c_js over (c+_i, c+_k, c~_l, c~_j)."""
    m = _invariant_one_body()
    return {(q1, q2, q3, q4): m[(q1, q4)] * m[(q2, q3)]
            for (q1, q4) in m for (q2, q3) in m}


def _group_coupling(n, two_s, two_k):
    """K[(q_1..q_n)][Q]: coupling of n rank-1/2 tensors on one subsystem to rank k with
    internal pair spin S: n=2 [T1xT2]^S; n=3 [[T1xT2]^S x T3]^k; n=4 [[T1xT2]^S x [T3xT4]^S]^k."""
    out = {}
    for qs in itertools.product(_HALF, repeat=n):
        if n == 0:
            out[qs] = {0: 1.0}
        elif n == 1:
            out[qs] = {qs[0]: 1.0}
        elif n == 2:
            w = cg(1, qs[0], 1, qs[1], two_s, qs[0] + qs[1])
            out[qs] = {qs[0] + qs[1]: w}
        elif n == 3:
            q12 = qs[0] + qs[1]
            w = cg(1, qs[0], 1, qs[1], two_s, q12) * cg(two_s, q12, 1, qs[2], two_k, q12 + qs[2])
            out[qs] = {q12 + qs[2]: w}
        else:
            q12, q34 = qs[0] + qs[1], qs[2] + qs[3]
            w = (cg(1, qs[0], 1, qs[1], two_s, q12) * cg(1, qs[2], 1, qs[3], two_s, q34)
                 * cg(two_s, q12, two_s, q34, two_k, q12 + q34))
            out[qs] = {q12 + q34: w}
    return out


def _group_options(n):
    """(two_S internal, two_k) choices for a subsystem holding n rank-1/2 operators."""
    if n == 0:
        return [(0, 0)]
    if n == 1:
        return [(0, 1)]
    if n == 2:
        return [(0, 0), (2, 2)]
    if n == 3:
        return [(0, 1), (2, 1), (2, 3)]
    return [(0, 0), (2, 0)]


_scheme_cache = {}


def _schemes(counts):
    """All coupling schemes for `counts` = (n_l, n_B, n_C, n_r): list of
    ((S_l,k_l),(S_B,k_B),(S_C,k_C),(S_r,k_r),k1, W) with W[q_all] the scheme tensor."""
    if counts in _scheme_cache:
        return _scheme_cache[counts]
    res = []
    for opts in itertools.product(*[_group_options(n) for n in counts]):
        (sl, kl), (sb, kb), (sc, kc), (sr, kr) = opts
        ks = [k for k in range(abs(kl - kb), kl + kb + 1, 2) if abs(kc - kr) <= k <= kc + kr and (k + kc + kr) % 2 == 0]
        if not ks:
            continue
        grp = [_group_coupling(n, s, k) for n, (s, k) in zip(counts, opts)]
        for k1 in ks:
            w = {}
            for ql in itertools.product(_HALF, repeat=counts[0]):
                for qb in itertools.product(_HALF, repeat=counts[1]):
                    for qc in itertools.product(_HALF, repeat=counts[2]):
                        for qr in itertools.product(_HALF, repeat=counts[3]):
                            tot = 0.0
                            for QL, wl in grp[0][ql].items():
                                for QB, wb in grp[1][qb].items():
                                    for QC, wc in grp[2][qc].items():
                                        for QR, wr in grp[3][qr].items():
                                            tot += (wl * wb * wc * wr
                                                    * cg(kl, QL, kb, QB, k1, QL + QB)
                                                    * cg(kc, QC, kr, QR, k1, QC + QR)
                                                    * cg(k1, QL + QB, k1, QC + QR, 0, 0))
                            if tot != 0.0:
                                w[ql + qb + qc + qr] = tot
            if w:
                res.append((opts, k1, w))
    _scheme_cache[counts] = res
    return res


def _elementary_rows(t, v, sub_of):
    """Steps 1-3: list of (alpha, (desc_l, desc_B, desc_C, desc_r), k1) with
    desc_X = (kinds, orbitals, two_S_internal, two_k)."""
    n = t.shape[0]
    rows = []
    inv1, inv2 = _invariant_one_body(), _invariant_two_body()

    def emit(coef, ops, inv):
        order = sorted(range(len(ops)), key=lambda a: sub_of[ops[a][1]])      # stable
        inversions = sum(1 for a in range(len(order)) for b in range(a + 1, len(order)) if order[a] > order[b])
        sign = -1.0 if inversions % 2 else 1.0
        sorted_ops = [ops[a] for a in order]
        counts = tuple(sum(1 for o in sorted_ops if sub_of[o[1]] == x) for x in range(4))
        iperm = {tuple(q[a] for a in order): val for q, val in inv.items()}
        norm2 = 0.0
        for opts, k1, w in _schemes(counts):
            alpha = sum(w.get(q, 0.0) * val for q, val in iperm.items())
            norm2 += alpha * alpha
            if abs(alpha) < 1e-14:
                continue
            descs, pos = [], 0
            for x in range(4):
                grp = sorted_ops[pos:pos + counts[x]]
                pos += counts[x]
                descs.append((tuple(o[0] for o in grp), tuple(o[1] for o in grp), opts[x][0], opts[x][1]))
            rows.append((coef * sign * alpha, tuple(descs), k1))
        assert abs(norm2 - sum(val * val for val in inv.values())) < 1e-12, "coupling schemes incomplete"

    for i in range(n):
        for j in range(n):
            if t[i, j] != 0.0:
                emit(t[i, j], [("+", i), ("~", j)], inv1)
    for i, j, k, l in itertools.product(range(n), repeat=4):
        if v[i, j, k, l] != 0.0:
            emit(0.5 * v[i, j, k, l], [("+", i), ("+", k), ("~", l), ("~", j)], inv2)
    return rows


class _Subsystem:
    def __init__(self, orbitals, is_site, keep=None):
        self.orbitals = list(orbitals)
        self.fs = FockSpace(len(self.orbitals))
        self.basis = site_multiplet_basis(self.fs) if is_site else full_multiplet_basis(self.fs)
        if keep is not None:
            self.basis = truncate_basis(self.basis, keep)
        self._cache = {}

    def tensor(self, desc):
        """TensorOp of the coupled product described by desc, in the local Fock space."""
        kinds, orbs, two_s, two_k = desc
        el = [self.fs.t_cd(self.orbitals.index(o)) if kd == "+" else self.fs.t_ct(self.orbitals.index(o))
              for kd, o in zip(kinds, orbs)]
        if len(el) == 0:
            return self.fs.t_identity()
        if len(el) == 1:
            return el[0]
        if len(el) == 2:
            return couple(el[0], el[1], two_s)
        if len(el) == 3:
            return couple(couple(el[0], el[1], two_s), el[2], two_k)
        return couple(couple(el[0], el[1], two_s), couple(el[2], el[3], two_s), two_k)

    def reduced(self, desc):
        if desc not in self._cache:
            self._cache[desc] = reduce_tensor(self.tensor(desc), self.basis)
        return self._cache[desc]


def _add_blocks(acc, blocks, scale):
    for key, m in blocks.items():
        if key in acc:
            acc[key] = acc[key] + scale * m
        else:
            acc[key] = scale * m


def _site_canonical(red):
    """Canonical representative of a site operator up to scale: (3x3 table / first non-zero, scale)."""
    r = np.zeros((3, 3))
    for (o, i), m in red.items():
        r[o, i] = m[0, 0]
    nz = np.flatnonzero(np.abs(r.ravel()) > 1e-13)
    if len(nz) == 0:
        return None, 0.0
    lam = r.ravel()[nz[0]]
    return r / lam, lam


def build_problem(t, v, n_left, n_elec, two_s_tot, keep_l=None, keep_r=None, use_adjoints=False, drop_tol=1e-14,
                  decomposition=None):
    """Exact `Problem` for the superblock l=[0,n_left) | B=n_left | C=n_left+1 | r=rest.

    decomposition: if a dict is passed, it receives for every pre-contracted ("complementary") family the ingredients of
    its pre-contraction, decomposition[(side, family index)] = (normal, W): `normal` is the family of the
    NORMAL operators of that block the complementary ones are made of (one position per distinct coupled product of
    elementary operators), W[pos', pos] the integral-dependent weight of normal operator pos in complementary operator
    pos' -- so that family[pos'] = sum_pos W[pos', pos] normal[pos], which is how this module itself accumulates them."""
    t = np.asarray(t, dtype=float)
    v = np.asarray(v, dtype=float)
    n_orb = t.shape[0]
    sub_of = [0] * n_left + [1, 2] + [3] * (n_orb - n_left - 2)
    subs = [_Subsystem(range(0, n_left), False, keep_l), _Subsystem([n_left], True),
            _Subsystem([n_left + 1], True), _Subsystem(range(n_left + 2, n_orb), False, keep_r)]

    # step 4: merge identical rows, then pre-contract over the block with more operators
    merged = {}
    for alpha, descs, k1 in _elementary_rows(t, v, sub_of):
        key = (descs, k1)
        merged[key] = merged.get(key, 0.0) + alpha

    site_ops, site_index = [], {}

    def site_id(x, desc):
        red = subs[x].reduced(desc)
        canon, lam = _site_canonical(red)
        if canon is None:
            return None, 0.0
        dN = sum(+1 if kd == "+" else -1 for kd in desc[0])
        key = (dN, desc[3], tuple(np.round(canon.ravel(), 12)))
        if key not in site_index:
            site_index[key] = len(site_ops)
            site_ops.append(SiteOp(dN=dN, twoK=desc[3], r=canon.copy(), name="site%d" % len(site_ops)))
        return site_index[key], lam

    # groups[(side, normal desc, opB, opC, k1, (dN, two_k) of contracted op)] -> reduced blocks
    groups, raw = {}, {}
    for (descs, k1), alpha in merged.items():
        if abs(alpha) < drop_tol:
            continue
        dl, db, dc, dr = descs
        ob, lb = site_id(1, db)
        oc, lc = site_id(2, dc)
        if ob is None or oc is None:
            continue
        a = alpha * lb * lc
        contract_r = len(dl[0]) <= len(dr[0])
        nd, cd_, cx = (dl, dr, 3) if contract_r else (dr, dl, 0)
        cdn = sum(+1 if kd == "+" else -1 for kd in cd_[0])
        gkey = ("r" if contract_r else "l", nd, ob, oc, k1, (cdn, cd_[3]))
        _add_blocks(groups.setdefault(gkey, {}), subs[cx].reduced(cd_), a)
        raw.setdefault(gkey, []).append((cd_, a))

    # step 5: families.  Normal operators of one type (kinds, S, k) form a family whose
    # positions are the orbital tuples; each group contributes one position of a
    # complementary family on the other block.
    normal_fams = {"l": {}, "r": {}}      # type key -> {orbitals: blocks}
    for (side, nd, ob, oc, k1, ck), blocks in groups.items():
        nside = "l" if side == "r" else "r"
        if len(nd[0]) == 0:
            continue
        tkey = (nd[0], nd[2], nd[3])
        normal_fams[nside].setdefault(tkey, {})[nd[1]] = subs[0 if nside == "l" else 3].reduced(nd)

    def make_family(pos_blocks, dN, two_k, secs, name):
        """pos_blocks: list (one per position) of {(io,ii): matrix}."""
        keys = sorted({k for pb in pos_blocks for k in pb})
        data = []
        for (io, ii) in keys:
            arr = np.zeros((len(pos_blocks), secs[io].dim, secs[ii].dim))
            for p, pb in enumerate(pos_blocks):
                if (io, ii) in pb:
                    arr[p] = pb[(io, ii)]
            data.append(arr)
        return OpFamily(dN=dN, twoK=two_k, npos=len(pos_blocks), q_out=[k[0] for k in keys],
                        q_in=[k[1] for k in keys], data=data, name=name)

    sec_l = [Sector(*s) for s in subs[0].basis.sectors]
    sec_r = [Sector(*s) for s in subs[3].basis.sectors]
    fams = {"l": [], "r": []}
    secs = {"l": sec_l, "r": sec_r}
    normal_id, normal_pos = {"l": {}, "r": {}}, {"l": {}, "r": {}}
    for side in ("l", "r"):
        for tkey in sorted(normal_fams[side], key=repr):
            orbs = sorted(normal_fams[side][tkey])
            dN = sum(+1 if kd == "+" else -1 for kd in tkey[0])
            fam = make_family([normal_fams[side][tkey][o] for o in orbs], dN, tkey[2], secs[side],
                              "N%s%s" % (side, tkey))
            normal_id[side][tkey] = len(fams[side])
            normal_pos[side][tkey] = orbs
            fams[side].append(fam)

    # terms: one per (contract side, normal type, opB, opC, k1, contracted type)
    term_groups = {}
    for (side, nd, ob, oc, k1, ck), blocks in groups.items():
        tkey = (nd[0], nd[2], nd[3]) if len(nd[0]) else None
        term_groups.setdefault((side, tkey, ob, oc, k1, ck), {})[nd[1]] = blocks
    terms = []
    for (side, tkey, ob, oc, k1, ck) in sorted(term_groups, key=repr):
        nside = "l" if side == "r" else "r"
        by_orb = term_groups[(side, tkey, ob, oc, k1, ck)]
        if tkey is None:
            pos_blocks = [by_orb[()]]
            nfam = -1
        else:
            pos_blocks = [by_orb.get(o, {}) for o in normal_pos[nside][tkey]]
            nfam = normal_id[nside][tkey]
        if all(len(pb) == 0 or max(np.abs(m).max() for m in pb.values()) < drop_tol for pb in pos_blocks):
            continue
        cfam = make_family(pos_blocks, ck[0], ck[1], secs[side], "C%s%s" % (side, (tkey, ob, oc, k1)))
        cid = len(fams[side])
        fams[side].append(cfam)
        if decomposition is not None:
            orbs_list = [()] if tkey is None else normal_pos[nside][tkey]
            lists = [raw.get((side, (() if tkey is None else tkey[0], o, 0 if tkey is None else tkey[1],
                                     0 if tkey is None else tkey[2]), ob, oc, k1, ck), []) for o in orbs_list]
            descs_in = sorted({d for lst in lists for d, _ in lst}, key=repr)
            w = np.zeros((len(orbs_list), len(descs_in)))
            for p, lst in enumerate(lists):
                for d, a in lst:
                    w[p, descs_in.index(d)] += a
            cx = 3 if side == "r" else 0
            normal = make_family([subs[cx].reduced(d) for d in descs_in], ck[0], ck[1], secs[side], "normal of " + cfam.name)
            decomposition[(side, cid)] = (normal, w)
        fam_l, fam_r = (nfam, cid) if side == "r" else (cid, nfam)
        terms.append(Term(fam_l=fam_l, fam_r=fam_r, op_B=ob, op_C=oc, twoK_L=k1, twoK_R=k1,
                          name="%s|%s" % (side, tkey)))

    prob = Problem(n_tot=n_elec, twoS_tot=two_s_tot, sec_l=sec_l, sec_r=sec_r, fam_l=fams["l"], fam_r=fams["r"],
                   site=site_ops, term=terms, meta={"n_orb": n_orb, "n_left": n_left})
    if use_adjoints:
        _replace_by_adjoints(prob, subs)
    return prob


def _adjoint_blocks(fam, secs):
    """Reduced blocks of the adjoint tensor of a family, DIRECTLY from the definition
    T~_q = (-1)^(k+q) (T_{-q})^dagger evaluated with Clebsch-Gordan coefficients (no C1.8):
    <S'||T~||S> = (-1)^(k+q) <k -q; S M|S' M'> / <k q; S' M'... > -- done numerically per block."""
    out = {}
    k = fam.twoK
    for b, (qo, qi) in enumerate(zip(fam.q_out, fam.q_in)):
        so, si = secs[qo].twoS, secs[qi].twoS
        # adjoint maps sector qo -> qi.  Pick M = so (ket), q with M' = so + q valid.
        ratio = None
        for q in range(-k, k + 1, 2):
            mp = so + q
            if abs(mp) > si:
                continue
            den = cg(k, q, so, so, si, mp)                      # <k q; S M|S' M'> for T~ (convention B)
            num = (-1) ** ((k + q) // 2) * cg(k, -q, si, mp, so, so)  # (-1)^(k+q) <S M|T_{-q}|S' M'>*
            if abs(den) > 1e-12:
                ratio = num / den
                break
        out[(qi, qo)] = ratio * np.swapaxes(fam.data[b], 1, 2)
    return out


def _replace_by_adjoints(prob, subs):
    """Where a family G equals lam * adjoint-tensor(F) of another family F of the same block
    (position by position), use (F, adj=1, alpha*=lam) instead of G in the terms."""
    for side, fams, secs in (("l", prob.fam_l, prob.sec_l), ("r", prob.fam_r, prob.sec_r)):
        repl = {}
        for gi, g in enumerate(fams):
            gb = {(qo, qi): g.data[b] for b, (qo, qi) in enumerate(zip(g.q_out, g.q_in))}
            for fi, f in enumerate(fams):
                if fi == gi or fi in repl or f.npos != g.npos or f.twoK != g.twoK or f.dN != -g.dN:
                    continue
                if f.dN < 0 or (f.dN == 0 and fi > gi):
                    continue
                adj = _adjoint_blocks(f, secs)
                if set(adj) != set(gb):
                    continue
                num = sum(float((adj[kk] * gb[kk]).sum()) for kk in adj)
                den = sum(float((adj[kk] ** 2).sum()) for kk in adj)
                if den == 0.0:
                    continue
                lam = num / den
                err = sum(float(((gb[kk] - lam * adj[kk]) ** 2).sum()) for kk in adj)
                if abs(lam) > 1e-12 and err < 1e-22 * den:
                    repl[gi] = (fi, lam)
                    break
        for tm in prob.term:
            fam = tm.fam_l if side == "l" else tm.fam_r
            if fam in repl:
                fi, lam = repl[fam]
                npos = prob.npos_of(tm)
                a = np.ones(npos) if tm.alpha is None else np.asarray(tm.alpha, dtype=float)
                tm.alpha = a * lam
                if side == "l":
                    tm.fam_l, tm.adj_l = fi, 1
                else:
                    tm.fam_r, tm.adj_r = fi, 1
        prob.meta["adjoint_replacements_" + side] = len(repl)
