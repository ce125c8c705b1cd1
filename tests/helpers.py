"""Test helpers: glue between the oracle's dict-of-blocks and the plan's flat Psi layout, and a
throw-away host walk of the plan's task table (isolates planner bugs from kernel bugs)."""
import numpy as np

from oracle.heff_dense import heff_apply


def oracle_flat(problem, plan, psi_flat, terms=None):
    """F = H_eff psi by the oracle, in the plan's flat layout."""
    psi_red = {}
    for lab, o0, o1 in zip(plan.labels, plan.offsets[:-1], plan.offsets[1:]):
        m, n = problem.sec_l[lab[0]].dim, problem.sec_r[lab[4]].dim
        psi_red[lab] = np.asarray(psi_flat[o0:o1]).reshape(m, n)
    f = heff_apply(problem, psi_red, terms=terms)
    assert set(f) == set(plan.labels)
    return np.concatenate([f[lab].ravel() for lab in plan.labels])


def host_walk(problem, plan, psi_flat):
    """Walk the exported task table with numpy: F_s += coef sum_pos alpha A E D^T."""
    t = plan.export_tasks()
    out = np.zeros(plan.psi_len)
    for i in range(len(t["coef"])):
        so, si = t["out_sec"][i], t["in_sec"][i]
        lo, li = plan.labels[so], plan.labels[si]
        m, p = problem.sec_l[lo[0]].dim, problem.sec_r[lo[4]].dim
        k, n = problem.sec_l[li[0]].dim, problem.sec_r[li[4]].dim
        e = psi_flat[plan.offsets[si]:plan.offsets[si + 1]].reshape(k, n)
        term = problem.term[t["term"][i]]
        npos = problem.npos_of(term)
        alpha = np.ones(npos) if term.alpha is None else np.asarray(term.alpha)

        def blocks(fams, fam, blk, adj, dim):
            if fam < 0:
                return np.eye(dim)[None]
            a = fams[fam].data[blk]
            return np.swapaxes(a, 1, 2) if adj else a
        a = blocks(problem.fam_l, t["fam_l"][i], t["blk_l"][i], t["adj_l"][i], m)
        d = blocks(problem.fam_r, t["fam_r"][i], t["blk_r"][i], t["adj_r"][i], p)
        acc = np.zeros((m, p))
        for pos in range(npos):
            ap = a[pos if a.shape[0] > 1 else 0]
            dp = d[pos if d.shape[0] > 1 else 0]
            acc += alpha[pos] * (ap @ e @ dp.T)
        out[plan.offsets[so]:plan.offsets[so + 1]] += t["coef"][i] * acc.ravel()
    return out
