"""Pins P8, P9, P10: the whole oracle chain
integrals -> exact operator table -> M-resolved H_eff Psi -> reduced result
against exact diagonalisation of the Jordan-Wigner Hamiltonian."""
import numpy as np
import pytest

from gen.workloads import CONFIGS, config_problem, integrals
from oracle.abinitio_table import build_problem
from oracle.fock import FockSpace
from oracle.heff_dense import flatten, heff_apply, heff_matrix, psi_sectors, unflatten
from test_oracle_fock import heisenberg_integrals, sector_spectrum


def _random_integrals(n, seed):
    rng = np.random.default_rng(seed)
    t = rng.normal(size=(n, n))
    t = (t + t.T) / 2
    v = rng.normal(size=(n, n, n, n))
    v = v + v.transpose(1, 0, 2, 3)
    v = v + v.transpose(0, 1, 3, 2)
    v = v + v.transpose(2, 3, 0, 1)
    return t, v


@pytest.mark.parametrize("L,nl,N,twoS", [(4, 1, 4, 0), (4, 1, 3, 1), (4, 1, 4, 2), (5, 2, 5, 1), (5, 1, 4, 0)])
def test_heff_spectrum_equals_fci_untruncated(L, nl, N, twoS):
    """P9: with complete blocks H_eff IS the Hamiltonian of the (N,S) sector."""
    t, v = _random_integrals(L, 11 + L)
    prob = build_problem(t, v, nl, N, twoS)
    h = heff_matrix(prob)
    assert np.abs(h - h.T).max() < 1e-12
    fs = FockSpace(L)
    ref = sector_spectrum(fs, fs.hamiltonian(t, v), N, twoS)
    assert h.shape[0] == len(ref)
    assert np.abs(np.linalg.eigvalsh((h + h.T) / 2) - ref).max() < 1e-10


def test_cfg1_spectrum_equals_fci():
    """P9 at BASELINE.json configs[0]: L=6, N=6, S=0, D_SU2=16 >= the 10 multiplets of a
    2-orbital block, so the blocks are complete: 53 Psi sectors, 175 elements = W(6,6,0)."""
    c = CONFIGS["cfg1"]
    t, v = integrals(c["L"], seed=0, xi=c["xi"])
    prob = build_problem(t, v, 2, c["N"], c["twoS"])
    assert [(s.N, s.twoS, s.dim) for s in prob.sec_l] == [(0, 0, 1), (1, 1, 2), (2, 0, 3), (2, 2, 1), (3, 1, 2), (4, 0, 1)]
    labels = psi_sectors(prob)
    assert len(labels) == 53
    h = heff_matrix(prob)
    assert h.shape == (175, 175)
    assert np.abs(h - h.T).max() < 1e-13
    fs = FockSpace(6)
    ref = sector_spectrum(fs, fs.hamiltonian(t, v), 6, 0)
    assert len(ref) == 175
    assert np.abs(np.linalg.eigvalsh((h + h.T) / 2) - ref).max() < 1e-11


def test_adjoint_flags_reproduce_explicit_families():
    """The oracle's handling of Term.adj_l/adj_r (definition T~_q = (-1)^(k+q)(T_-q)^dagger):
    replacing c~ families by adjoint(c+) leaves H_eff unchanged."""
    t, v = _random_integrals(5, 3)
    p0 = build_problem(t, v, 2, 5, 1)
    p1 = build_problem(t, v, 2, 5, 1, use_adjoints=True)
    assert p1.meta["adjoint_replacements_l"] + p1.meta["adjoint_replacements_r"] > 0
    assert any(tm.adj_l or tm.adj_r for tm in p1.term)
    rng = np.random.default_rng(0)
    n = len(flatten(p0, {}))
    x = rng.normal(size=n)
    f0 = flatten(p0, heff_apply(p0, unflatten(p0, x)))
    f1 = flatten(p1, heff_apply(p1, unflatten(p1, x)))
    assert np.abs(f0 - f1).max() < 1e-12 * np.abs(f0).max()


def test_heisenberg_ring_through_the_whole_chain():
    """P8: 4-site Heisenberg ring, one orbital per subsystem, (N=4, S=0): E0 = -2J."""
    J = 0.7
    t, v = heisenberg_integrals(4, [(0, 1), (1, 2), (2, 3), (3, 0)], J)
    h = heff_matrix(build_problem(t, v, 1, 4, 0))
    w = np.linalg.eigvalsh((h + h.T) / 2)
    assert abs(w[0] + 2 * J) < 1e-12
    # dimer on the two sites only (blocks empty of electrons are still present): singlet -3J/4
    t2, v2 = heisenberg_integrals(4, [(1, 2)], J)
    h2 = heff_matrix(build_problem(t2, v2, 1, 2, 0))
    assert abs(np.linalg.eigvalsh((h2 + h2.T) / 2)[0] + 0.75 * J) < 1e-12


def test_truncated_blocks_give_projected_hamiltonian():
    """With truncated (rotated) block bases H_eff = P H P: its spectrum interlaces, and
    its lowest eigenvalue is variational (>= FCI)."""
    t, v = _random_integrals(5, 5)
    from oracle.multiplets import full_multiplet_basis
    rng = np.random.default_rng(1)
    keep = {}
    for isec, (n, s, d) in enumerate(full_multiplet_basis(FockSpace(2)).sectors):
        q, _ = np.linalg.qr(rng.normal(size=(d, d)))
        keep[isec] = q[:, :max(1, d - 1)]
    prob = build_problem(t, v, 2, 5, 1, keep_l=keep)
    h = heff_matrix(prob)
    assert np.abs(h - h.T).max() < 1e-12
    fs = FockSpace(5)
    ref = sector_spectrum(fs, fs.hamiltonian(t, v), 5, 1)
    w = np.linalg.eigvalsh((h + h.T) / 2)
    assert len(w) < len(ref)
    assert w[0] >= ref[0] - 1e-10
    assert w[-1] <= ref[-1] + 1e-10
    for i in range(len(w)):                       # Cauchy interlacing
        assert ref[i] - 1e-10 <= w[i] <= ref[i + len(ref) - len(w)] + 1e-10


def test_synthetic_workload_is_hermitian_and_scalar():
    """P10 on the random-operator generator (every row has its Hermitian conjugate):
    <phi|H psi> = <H phi|psi>; heff_apply itself checks the leakage invariant O6."""
    prob = config_problem("mini")
    n = len(flatten(prob, {}))
    rng = np.random.default_rng(0)
    x, y = rng.normal(size=n), rng.normal(size=n)
    hx = flatten(prob, heff_apply(prob, unflatten(prob, x)))
    hy = flatten(prob, heff_apply(prob, unflatten(prob, y)))
    assert abs(y @ hx - x @ hy) < 1e-11 * abs(y @ hx)
    z = flatten(prob, heff_apply(prob, unflatten(prob, 2.0 * x - 0.5 * y)))
    assert np.abs(z - (2.0 * hx - 0.5 * hy)).max() < 1e-11 * np.abs(hx).max()


def test_rank_mismatched_row_vanishes():
    """A row with k1 != k2 cannot be coupled to rank 0 ("k=0 as the Hamilton
    is a spin zero object"): its contribution is identically zero."""
    prob = config_problem("mini")
    bad = [tm for tm in prob.term if tm.name == "B1Q1"][0]
    bad.fam_r = [i for i, f in enumerate(prob.fam_r) if f.name == "Q0(r)"][0]
    bad.twoK_R = 0
    n = len(flatten(prob, {}))
    x = np.random.default_rng(0).normal(size=n)
    f = flatten(prob, heff_apply(prob, unflatten(prob, x), terms=[bad]))
    assert np.abs(f).max() == 0.0


def test_sampled_equals_full_oracle():
    """oracle/heff_sampled.py (step O7: sampled entries for the large configs) against the full
    M-resolved oracle on workloads where both run: exact cfg1 Hamiltonian and the random 'mini' table."""
    from gen.workloads import config_problem, integrals, random_psi
    from oracle.abinitio_table import build_problem
    from oracle.heff_dense import flatten, heff_apply, psi_sectors, unflatten
    from oracle.heff_sampled import heff_sample, numpy_block_rows
    t, v = integrals(6, seed=0, xi=2.0)
    for prob in (build_problem(t, v, 2, 6, 0, use_adjoints=True), config_problem("mini")):
        labels = psi_sectors(prob)
        n = sum(prob.sec_l[s[0]].dim * prob.sec_r[s[4]].dim for s in labels)
        psi = unflatten(prob, random_psi(n, seed=3), labels)
        ref = heff_apply(prob, psi)
        rows = numpy_block_rows(prob)
        rng = np.random.default_rng(1)
        checked = 0
        for lab in labels[::5]:
            m, p = prob.sec_l[lab[0]].dim, prob.sec_r[lab[4]].dim
            ra = np.sort(rng.choice(m, size=min(m, 3), replace=False))
            rb = np.sort(rng.choice(p, size=min(p, 2), replace=False))
            got = heff_sample(prob, psi, lab, ra, rb, rows)
            want = ref[lab][np.ix_(ra, rb)]
            assert np.abs(got - want).max() <= 1e-13 * max(1.0, np.abs(flatten(prob, ref, labels)).max())
            checked += got.size
        assert checked > 20


def _position_loop(a, d, alpha, e, rows_a, rows_b):
    """sum_pos alpha_pos A_pos[rows_a, :] E D_pos[rows_b, :]^T with python loops over every index
    (PAPER.md:58-60); a / d: [npos or 1, m, k] / [npos or 1, p, n] full applied blocks or None (identity)."""
    out = np.zeros((len(rows_a), len(rows_b)))
    k, n = e.shape
    for pos in range(len(alpha)):
        ap = np.eye(k) if a is None else a[pos if a.shape[0] > 1 else 0]
        dp = np.eye(n) if d is None else d[pos if d.shape[0] > 1 else 0]
        for ia, ra in enumerate(rows_a):
            for ib, rb in enumerate(rows_b):
                s = 0.0
                for x in range(k):
                    for y in range(n):
                        s += ap[ra, x] * e[x, y] * dp[rb, y]
                out[ia, ib] += alpha[pos] * s
    return out


def test_sampled_sum_equals_position_loop():
    """Pins the position sum of BOTH oracles (heff_dense._sum_over_positions, heff_sampled._sampled_sum) against
    scalar loops on random blocks with non-trivial alpha, for every combination of operands that varies with
    the position, is fixed (one position), or is the identity -- including len(alpha) > 1 with neither varying."""
    from types import SimpleNamespace
    from oracle.heff_dense import _sum_over_positions
    from oracle.heff_sampled import _sampled_sum
    rng = np.random.default_rng(5)
    m, k, n, p, npos = 4, 5, 3, 6, 7
    e = rng.normal(size=(k, n))
    alpha = rng.normal(size=npos) + 0.3
    rows = {"m": np.array([0, 2, 3]), "p": np.array([1, 4])}
    kinds = ("varies", "fixed", "identity")
    for ka in kinds:
        for kd in kinds:
            for tr in (False, True):
                mm = k if ka == "identity" else m
                pp = n if kd == "identity" else p
                a = None if ka == "identity" else rng.normal(size=(npos if ka == "varies" else 1, mm, k))
                d = None if kd == "identity" else rng.normal(size=(npos if kd == "varies" else 1, pp, n))
                ra = rows["m"][rows["m"] < mm]
                rb = rows["p"][rows["p"] < pp]
                want = _position_loop(a, d, alpha, e, ra, rb)
                got_s = _sampled_sum(None if a is None else a[:, ra, :], None if d is None else d[:, rb, :], alpha, e, ra, rb)
                assert np.abs(got_s - want).max() < 1e-13
                # the dense oracle takes STORED blocks + adjoint flags: store the transposes when tr is set
                fl = None if a is None else SimpleNamespace(data=[np.swapaxes(a, 1, 2).copy() if tr else a])
                fr = None if d is None else SimpleNamespace(data=[np.swapaxes(d, 1, 2).copy() if tr else d])
                got_d = _sum_over_positions(fl, 0, tr, fr, 0, tr, alpha, e)
                assert np.abs(got_d[np.ix_(ra, rb)] - want).max() < 1e-13
                # batched E (heff_matrix pushes all unit vectors of a sector at once)
                got_b = _sum_over_positions(fl, 0, tr, fr, 0, tr, alpha, np.stack([e, 2.0 * e]))
                assert np.abs(got_b[1][np.ix_(ra, rb)] - 2.0 * want).max() < 1e-13
