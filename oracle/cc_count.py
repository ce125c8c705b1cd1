"""ORACLE-side test infrastructure (never imported by the product path).

The paper's measure of work, CC = "the sum of all the computational complexity ... to perform the sequence of matrix
and tensor operations according to Eq. (2)", for the reduced (SU(2)) sector tasks of a problem, counted
in plain Python from the sector tables: every (operator-table row, sector combination) whose recoupling coefficient is
non-zero contributes min(2mkn + 2mnp, 2knp + 2mkp) flops per position.  A row whose positions enter through one
block only is ONE position (its sum over positions is Psi-independent: DESIGN.md reading G13).

Used by bench.py's reference arm (which must not load the CUDA library) and pinned against the planner's own count
(su2_plan_info_t.cc_flops) in tests/test_planner_cpu.py::test_cc_count_matches_the_planner.
"""
from .heff_dense import SITE_2S, SITE_N, psi_sectors
from .wigner import c_hat


def cc_flops(problem):
    """(CC in flops, number of sector tasks, number of task-positions)."""
    labels = set(psi_sectors(problem))
    by_quad = {}
    for lab in labels:
        by_quad.setdefault((lab[0], lab[1], lab[3], lab[4]), []).append(lab)
    s_tot = problem.twoS_tot
    cc, ntask, ntp = 0.0, 0, 0
    for t in problem.term:
        fl = problem.fam_l[t.fam_l] if t.fam_l >= 0 else None
        fr = problem.fam_r[t.fam_r] if t.fam_r >= 0 else None
        oB, oC = problem.site[t.op_B], problem.site[t.op_C]
        kl = fl.twoK if fl is not None else 0
        kr = fr.twoK if fr is not None else 0
        k1, k2 = t.twoK_L, t.twoK_R
        npl = fl.npos if fl is not None else 1
        npr = fr.npos if fr is not None else 1
        npos = max(npl, npr)
        if npos > 1 and (npl > 1) != (npr > 1):
            npos = 1                                       # one-sided row: folded over its positions

        def transitions(fam, adj, secs):
            if fam is None:
                return [(i, i) for i in range(len(secs))]
            return [((qo, qi) if adj else (qi, qo)) for qo, qi in zip(fam.q_out, fam.q_in)]    # (ket, bra) of the applied operator
        for li, lo in transitions(fl, t.adj_l, problem.sec_l):
            for sBi in range(3):
                sBo = sBi + oB.dN
                if not 0 <= sBo <= 2 or oB.r[sBo][sBi] == 0.0:
                    continue
                for sCi in range(3):
                    sCo = sCi + oC.dN
                    if not 0 <= sCo <= 2 or oC.r[sCo][sCi] == 0.0:
                        continue
                    for ri, ro in transitions(fr, t.adj_r, problem.sec_r):
                        for a in by_quad.get((lo, sBo, sCo, ro), ()):
                            for b in by_quad.get((li, sBi, sCi, ri), ()):
                                Sl, Slp = problem.sec_l[lo].twoS, problem.sec_l[li].twoS
                                Sr, Srp = problem.sec_r[ro].twoS, problem.sec_r[ri].twoS
                                if c_hat(Sl, SITE_2S[sBo], a[2], kl, oB.twoK, k1, Slp, SITE_2S[sBi], b[2]) == 0.0:
                                    continue
                                if c_hat(SITE_2S[sCo], Sr, a[5], oC.twoK, kr, k2, SITE_2S[sCi], Srp, b[5]) == 0.0:
                                    continue
                                if c_hat(a[2], a[5], s_tot, k1, k2, 0, b[2], b[5], s_tot) == 0.0:
                                    continue
                                m, p = problem.sec_l[lo].dim, problem.sec_r[ro].dim
                                k, n = problem.sec_l[li].dim, problem.sec_r[ri].dim
                                cc += npos * min(2.0 * m * k * n + 2.0 * m * n * p, 2.0 * k * n * p + 2.0 * m * k * p)
                                ntask += 1
                                ntp += npos
    assert SITE_N == (0, 1, 2)
    return cc, ntask, ntp
