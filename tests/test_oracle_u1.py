"""Pins of the U(1)-only mode oracle (oracle/heff_u1.py) and of the planner's
U(1) mode (host walk of its task table, no GPU)."""
import numpy as np
import pytest

from gen.workloads import config_problem, integrals, random_psi
from oracle.abinitio_table import build_problem
from oracle.fock import FockSpace
from oracle.heff_dense import flatten, heff_apply, psi_sectors, unflatten
from oracle.heff_u1 import (expand_problem, expand_psi_u1, flatten_u1, heff_apply_u1, project_psi_u1, psi_sectors_u1,
                            unflatten_u1)


def _matrix_u1(u1):
    labels = psi_sectors_u1(u1)
    n = len(flatten_u1(u1, {}, labels))
    h = np.zeros((n, n))
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1.0
        h[:, j] = flatten_u1(u1, heff_apply_u1(u1, unflatten_u1(u1, e, labels)), labels)
    return h


@pytest.mark.parametrize("merged", [False, True])
def test_u1_oracle_spectrum_equals_fci_in_the_sz_sector(merged):
    """heff_apply_u1 on the expansion of the exact ab initio table (complete blocks): its matrix is the Jordan-Wigner
    Hamiltonian restricted to (N, S_z = S_tot), so its spectrum is the FCI spectrum of ALL total spins S >= S_z of that
    sector -- computed independently with oracle/fock.py."""
    L, nl, N, twoS = 4, 1, 4, 0
    rng = np.random.default_rng(5)
    t = rng.normal(size=(L, L)); t = (t + t.T) / 2
    v = rng.normal(size=(L, L, L, L))
    v = v + v.transpose(1, 0, 2, 3); v = v + v.transpose(0, 1, 3, 2); v = v + v.transpose(2, 3, 0, 1)
    prob = build_problem(t, v, nl, N, twoS)
    u1, _ = expand_problem(prob, merged=merged)
    h = _matrix_u1(u1)
    assert np.abs(h - h.T).max() < 1e-12
    fs = FockSpace(L)
    hfull = fs.hamiltonian(t, v)
    sel = fs.sector_indices(N, twoS)
    ref = np.linalg.eigvalsh(np.asarray(hfull[np.ix_(sel, sel)].todense()))
    assert h.shape[0] == len(ref)
    assert np.abs(np.linalg.eigvalsh((h + h.T) / 2) - ref).max() < 1e-10


@pytest.mark.parametrize("name,merged", [("cfg1x", False), ("cfg1x", True), ("mini", False), ("mini", True)])
def test_su2_result_is_the_u1_result_times_scalars(name, merged):
    """the SU(2) calculation is the U(1) one "modified only by constant multiplication factors": the
    reduced oracle result, expanded, equals the U(1) oracle on the expanded problem; projected back it is the same."""
    if name == "cfg1x":
        t, v = integrals(6, seed=0, xi=2.0)
        prob = build_problem(t, v, 2, 6, 0, use_adjoints=True)
    else:
        prob = config_problem(name)
    labels = psi_sectors(prob)
    n = sum(prob.sec_l[s[0]].dim * prob.sec_r[s[4]].dim for s in labels)
    psi = unflatten(prob, random_psi(n, seed=4), labels)
    f_red = heff_apply(prob, psi)
    u1, maps = expand_problem(prob, merged=merged)
    f_u1 = heff_apply_u1(u1, expand_psi_u1(prob, u1, maps, psi))
    want = expand_psi_u1(prob, u1, maps, f_red)
    scale = max(np.abs(b).max() for b in want.values())
    assert max(np.abs(f_u1[k] - want[k]).max() for k in want) <= 1e-12 * scale       # no leakage out of S_tot either
    back = project_psi_u1(prob, maps, f_u1)
    assert np.abs(flatten(prob, back, labels) - flatten(prob, f_red, labels)).max() <= 1e-12 * scale


@pytest.mark.parametrize("merged", [False, True])
def test_planner_u1_mode_task_table_equals_oracle(merged):
    """su2_plan_create with SU2_SYMMETRY_U1 (host-only): its Psi layout is psi_sectors_u1 and a numpy walk of its task
    table (unit recoupling factor: sign x site elements) equals heff_apply_u1."""
    from helpers import host_walk
    from paper_2309_16724_b200 import Plan
    prob = config_problem("mini")
    u1, _ = expand_problem(prob, merged=merged)
    plan = Plan(u1, host_only=True)
    labels = psi_sectors_u1(u1)
    assert plan.labels == labels
    x = random_psi(plan.psi_len, seed=2)
    ref = flatten_u1(u1, heff_apply_u1(u1, unflatten_u1(u1, x, labels)), labels)
    got = host_walk(u1, plan, x)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    # the ratio the paper's Table I reports: U(1) work over SU(2) work for the same operator
    su2 = Plan(prob, host_only=True)
    assert plan.info["cc_flops"] > su2.info["cc_flops"]
