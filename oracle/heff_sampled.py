"""ORACLE (test infrastructure only; never imported by the product path).

Sampled H_eff * Psi for workloads whose full oracle is too slow (SURVEY.md 8(c) C4 step O7,
BASELINE.json configs[2], configs[3]): the entries F_red[label][rows_a x rows_b] of ONE output sector,
computed by exactly the same M-resolved definition as oracle/heff_dense.py (O2-O6: Clebsch-Gordan
expansion of Psi, component-by-component application of every operator-table row with the
Jordan-Wigner signs, projection back) -- only restricted to the sampled rows of the left operator
blocks and the sampled rows of the right operator blocks, which is all those entries depend on:

    F_full[okey][a, b] = sum_rows coef * sum_pos alpha_pos * A_pos[a, :] E D_pos[b, :]^T .

Every operator-table row, every input sector and every position contributes; nothing is sampled
along the contraction.  Operator values are obtained through a callback so that blocks resident on a
device (92 GB at configs[3]) need not be staged through host memory in full.

Pins: tests/test_oracle_heff.py::test_sampled_equals_full_oracle (equality with heff_dense.heff_apply
on workloads small enough for both) and ::test_sampled_sum_equals_position_loop (the position sum against
scalar loops, every varying / fixed / identity operand combination, non-trivial alpha).
"""
import numpy as np

from .heff_dense import (SITE_2S, SITE_N, SITE_STATES, _block_element_factor, _block_transitions, _cg3,
                         _full_keys, expand_psi)
from .wigner import cg


def numpy_block_rows(problem):
    """block_rows callback for problems whose families carry numpy data."""
    def rows(side, fam_index, blk, idx, transposed):
        fam = (problem.fam_l if side == "l" else problem.fam_r)[fam_index]
        arr = fam.data[blk]
        if transposed:
            return np.swapaxes(arr[:, :, idx], 1, 2)
        return arr[:, idx, :]
    return rows


def heff_sample(problem, psi_red, label, rows_a, rows_b, block_rows, psi_full=None):
    """F_red[label][np.ix_(rows_a, rows_b)].

    block_rows(side, fam_index, blk, idx, transposed) -> array [npos, len(idx), inner]: rows `idx` of the
    APPLIED operator block (rows of the stored block, or its columns when the adjoint is applied)."""
    rows_a = np.asarray(rows_a, dtype=np.int64)
    rows_b = np.asarray(rows_b, dtype=np.int64)
    il_t, sB_t, j1_t, sC_t, ir_t, j2_t = label
    full = expand_psi(problem, psi_red) if psi_full is None else psi_full
    # M-resolved output components of the target sector and their projection weights (O6)
    want = {}
    for ml, b, c, mr, mb, mc in _full_keys(problem, label):
        w = _cg3(problem, label, ml, mb, mc, mr)
        if w != 0.0:
            want[(il_t, ml, b, c, ir_t, mr)] = w
    acc = {key: np.zeros((len(rows_a), len(rows_b))) for key in want}
    by_pair = {}                       # Psi_full components grouped by their (l sector, r sector)
    for key, blk in full.items():
        by_pair.setdefault((key[0], key[4]), []).append((key, blk))
    row_cache = {}

    def rows_of(side, fam_index, blk, idx, tr):
        key = (side, fam_index, blk, tr)
        if key not in row_cache:
            row_cache[key] = np.asarray(block_rows(side, fam_index, blk, idx, tr), dtype=np.float64)
        return row_cache[key]

    for t in problem.term:
        fl = problem.fam_l[t.fam_l] if t.fam_l >= 0 else None
        fr = problem.fam_r[t.fam_r] if t.fam_r >= 0 else None
        oB, oC = problem.site[t.op_B], problem.site[t.op_C]
        kl = fl.twoK if fl is not None else 0
        kr = fr.twoK if fr is not None else 0
        kB, kC = oB.twoK, oC.twoK
        k1, k2 = t.twoK_L, t.twoK_R
        dNr = 0 if fr is None else (-fr.dN if t.adj_r else fr.dN)
        pB, pC, pr = oB.dN & 1, oC.dN & 1, dNr & 1
        npos = problem.npos_of(t)
        alpha = np.ones(npos) if t.alpha is None else np.asarray(t.alpha, dtype=float)
        ltrans = [x for x in _block_transitions(fl, t.adj_l, problem.sec_l) if x[1] == il_t]
        rtrans = [x for x in _block_transitions(fr, t.adj_r, problem.sec_r) if x[1] == ir_t]
        if not ltrans or not rtrans:
            continue
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
                    for (li, lo, lb, ltr) in ltrans:
                        for (ri, ro, rb, rtr) in rtrans:
                            for key, blk in by_pair.get((li, ri), ()):
                                il_in, ml_in, b_in, c_in, ir_in, mr_in = key
                                sgb_in, mb_in = SITE_STATES[b_in]
                                sgc_in, mc_in = SITE_STATES[c_in]
                                sgb, sgc = sgb_in + oB.dN, sgc_in + oC.dN
                                if not (0 <= sgb <= 2 and 0 <= sgc <= 2):
                                    continue
                                mb, mc = mb_in + qB, mc_in + qC
                                eB = cg(kB, qB, SITE_2S[sgb_in], mb_in, SITE_2S[sgb], mb) * oB.r[sgb][sgb_in]
                                eC = cg(kC, qC, SITE_2S[sgc_in], mc_in, SITE_2S[sgc], mc) * oC.r[sgc][sgc_in]
                                if eB == 0.0 or eC == 0.0:
                                    continue
                                ml, mr = ml_in + ql, mr_in + qr
                                okey = (lo, ml, SITE_STATES.index((sgb, mb)), SITE_STATES.index((sgc, mc)), ro, mr)
                                if okey not in want:
                                    continue
                                s_li, s_lo = problem.sec_l[li].twoS, problem.sec_l[lo].twoS
                                s_ri, s_ro = problem.sec_r[ri].twoS, problem.sec_r[ro].twoS
                                el = 1.0 if fl is None else _block_element_factor(kl, ql, t.adj_l, s_li, ml_in, s_lo, ml)
                                er = 1.0 if fr is None else _block_element_factor(kr, qr, t.adj_r, s_ri, mr_in, s_ro, mr)
                                if el == 0.0 or er == 0.0:
                                    continue
                                n_l_in = problem.sec_l[il_in].N
                                sgn = (-1) ** (pB * n_l_in + pC * (n_l_in + SITE_N[sgb_in])
                                               + pr * (n_l_in + SITE_N[sgb_in] + SITE_N[sgc_in]))   # C1.7
                                a = None if fl is None else rows_of("l", t.fam_l, lb, rows_a, ltr)
                                d = None if fr is None else rows_of("r", t.fam_r, rb, rows_b, rtr)
                                acc[okey] += (w_op * eB * eC * sgn * el * er) * _sampled_sum(a, d, alpha, blk, rows_a, rows_b)
    out = np.zeros((len(rows_a), len(rows_b)))
    for key, w in want.items():
        out += w * acc[key]
    return out


def _sampled_sum(a, d, alpha, e, rows_a, rows_b):
    """sum_pos alpha_pos A_pos[rows_a, :] E D_pos[rows_b, :]^T; a: [npos or 1, |rows_a|, k] or None
    (identity), d: [npos or 1, |rows_b|, n] or None (identity).

    The same per-position terms as heff_dense._sum_over_positions, evaluated for all
    positions by ONE stacked call per product (np.matmul over a leading position axis) and then added
    with their alpha_pos: a family with a single position (or the identity) is repeated along that
    axis, never folded into the sum.  Pinned against the explicit position loop, for every
    combination of varying / fixed / identity operands and non-trivial alpha, by
    tests/test_oracle_heff.py::test_sampled_sum_equals_position_loop."""
    npos = len(alpha)
    if a is None:
        te = np.broadcast_to(e[rows_a, :], (npos,) + e[rows_a, :].shape)           # (1 E)[rows_a, :]
    else:
        # T_pos = A_pos[rows_a, :] E for every position: the position axis is stacked onto the row axis, so that all
        # positions share one library matmul ([npos * |rows_a|, k] @ [k, n]) -- the same products as the loop's
        stack = np.ascontiguousarray(np.broadcast_to(a, (npos,) + a.shape[1:]))
        te = np.matmul(stack.reshape(npos * a.shape[1], a.shape[2]), e).reshape(npos, a.shape[1], e.shape[1])
    if d is None:
        ted = te[:, :, rows_b]                                                      # (T_pos 1^T)[:, rows_b]
    else:
        ted = np.matmul(te, np.swapaxes(np.broadcast_to(d, (npos,) + d.shape[1:]), 1, 2))   # T_pos D_pos[rows_b, :]^T
    return np.tensordot(np.asarray(alpha, dtype=np.float64), ted, axes=(0, 0))      # sum_pos alpha_pos (...)
