"""Pins P3, P4, P6, P7, P8 for oracle/fock.py and oracle/multiplets.py."""
from math import sqrt

import numpy as np

from conftest import golden_lines
from gen.workloads import site_table, weyl_paldus
from oracle.fock import FockSpace, couple
from oracle.multiplets import full_multiplet_basis, reduce_tensor, site_multiplet_basis


def heisenberg_integrals(n, bonds, J):
    """J S_i.S_j per bond through 8-fold symmetric two-electron integrals (P8):
    (ij|ij)=(ij|ji)=(ji|ij)=(ji|ji) = -J/2, (ii|jj)=(jj|ii) = -J/4, t = 0."""
    v = np.zeros((n, n, n, n))
    for i, j in bonds:
        for a, b, c, d in ((i, j, i, j), (i, j, j, i), (j, i, i, j), (j, i, j, i)):
            v[a, b, c, d] += -J / 2
        v[i, i, j, j] += -J / 4
        v[j, j, i, i] += -J / 4
    return np.zeros((n, n)), v


def sector_spectrum(fs, h, n_elec, two_s):
    idx = fs.sector_indices(n_elec, two_s)
    hs = h[idx][:, idx].toarray()
    s2 = fs.s2()[idx][:, idx].toarray()
    w = np.linalg.eigvalsh(hs + 500.0 * (s2 - 0.25 * two_s * (two_s + 2) * np.eye(len(idx))))
    return w[w < 250.0]


def test_canonical_anticommutators():
    fs = FockSpace(2)
    ops = [fs.c(i, s) for i in range(2) for s in (0, 1)]
    for a, x in enumerate(ops):
        for b, y in enumerate(ops):
            assert abs(x @ y + y @ x).max() < 1e-15
            anti = (x @ y.T + y.T @ x).toarray()
            assert np.abs(anti - (np.eye(fs.dim) if a == b else 0)).max() < 1e-15
    # product state convention: creation operators in ascending mode order, sign +1
    vac = np.zeros(fs.dim)
    vac[0] = 1.0
    st = fs.cd(0, 0) @ (fs.cd(0, 1) @ (fs.cd(1, 1) @ vac))
    assert st[int("1101", 2)] == 1.0


def test_hubbard_dimer_closed_form():
    """P7: E0 = (U - sqrt(U^2 + 16 t^2))/2 at t = 1, U = 4."""
    fs = FockSpace(2)
    t = np.array([[0.0, -1.0], [-1.0, 0.0]])
    v = np.zeros((2, 2, 2, 2))
    v[0, 0, 0, 0] = v[1, 1, 1, 1] = 4.0
    w = sector_spectrum(fs, fs.hamiltonian(t, v), 2, 0)
    assert abs(w[0] - (4 - sqrt(16 + 16)) / 2) < 1e-12
    assert abs(w[0] + 0.8284271247461903) < 1e-12


def test_heisenberg_dimer_and_ring():
    """P8: dimer singlet -3J/4, triplet +J/4; 4-site ring ground state -2J."""
    J = 1.3
    fs = FockSpace(2)
    h = fs.hamiltonian(*heisenberg_integrals(2, [(0, 1)], J))
    assert abs(sector_spectrum(fs, h, 2, 0)[0] + 0.75 * J) < 1e-12
    assert abs(sector_spectrum(fs, h, 2, 2)[0] - 0.25 * J) < 1e-12
    fs4 = FockSpace(4)
    h4 = fs4.hamiltonian(*heisenberg_integrals(4, [(0, 1), (1, 2), (2, 3), (3, 0)], J))
    w = sector_spectrum(fs4, h4, 4, 0)
    assert abs(w[0] + 2 * J) < 1e-11


def test_elementary_tensors_are_spherical_tensors():
    """P3: [S_z, T_q] = q T_q, [S_+-, T_q] = sqrt((k-+q)(k+-q+1)) T_{q+-1}."""
    fs = FockSpace(2)
    sz, sp, sm = fs.sz(), fs.splus(), fs.sminus()
    cd0, ct1 = fs.t_cd(0), fs.t_ct(1)
    for op in (cd0, ct1, couple(cd0, ct1, 0), couple(cd0, ct1, 2), couple(cd0, fs.t_cd(1), 2),
               couple(couple(cd0, ct1, 2), fs.t_cd(1), 1), couple(couple(cd0, ct1, 2), fs.t_cd(1), 3)):
        k = op.two_k / 2
        for q2, m in op.comp.items():
            q = q2 / 2
            assert abs(sz @ m - m @ sz - q * m).max() < 1e-14
            up = sp @ m - m @ sp
            ref = sqrt((k - q) * (k + q + 1)) * op.comp[q2 + 2] if q2 + 2 in op.comp else 0 * m
            assert abs(up - ref).max() < 1e-14
            dn = sm @ m - m @ sm
            ref = sqrt((k + q) * (k - q + 1)) * op.comp[q2 - 2] if q2 - 2 in op.comp else 0 * m
            assert abs(dn - ref).max() < 1e-14


def _site_ops(fs):
    cd, ct = fs.t_cd(0), fs.t_ct(0)
    b0, b1 = couple(cd, ct, 0), couple(cd, ct, 2)
    nd = fs.cd(0, 0) @ fs.c(0, 0) @ fs.cd(0, 1) @ fs.c(0, 1)
    from oracle.fock import TensorOp
    return {"1": fs.t_identity(), "c+": cd, "c~": ct, "A0": couple(cd, cd, 0), "A~0": couple(ct, ct, 0),
            "B0": b0, "B1": b1, "B1c+": couple(b1, cd, 1), "B0c~": couple(b0, ct, 1), "D": TensorOp(0, 0, {0: nd})}


def test_site_table_golden_and_generator_table():
    """P4: brute-force reduction of the 4x4 site matrices reproduces tests/golden/site_table.txt
    (C1.6) and the table shipped in gen.workloads.site_table(), including its adjoint map."""
    fs = FockSpace(1)
    sb = site_multiplet_basis(fs)
    ops = _site_ops(fs)
    red = {name: {k: float(v[0, 0]) for k, v in reduce_tensor(op, sb).items()} for name, op in ops.items()}
    seen = {name: set() for name in ops}
    for name, o, i, *expr in golden_lines("site_table.txt"):
        val = eval(" ".join(expr))
        assert abs(red[name][(int(o), int(i))] - val) < 1e-14, name
        seen[name].add((int(o), int(i)))
    for name in ops:
        assert seen[name] == set(red[name])                 # no other non-zero element
    table, adj = site_table()
    for so in table:
        r = np.zeros((3, 3))
        for (o, i), val in red[so.name].items():
            r[o, i] = val
        assert np.abs(r - so.r).max() < 1e-14
        assert (so.dN, so.twoK) == (ops[so.name].dN, ops[so.name].two_k)
        # adjoint tensor T~_q = (-1)^(k+q) (T_-q)^dagger equals factor * partner
        partner, factor = adj[so.name]
        radj = {k: float(v[0, 0]) for k, v in reduce_tensor(ops[so.name].adjoint_tensor(), sb).items()}
        assert set(radj) == set(red[partner])
        for key, val in radj.items():
            assert abs(val - factor * red[partner][key]) < 1e-14


def test_multiplet_counts_weyl_paldus_and_adjoint_rule():
    """P6 (sector counting) and C1.8 (reduced elements of the adjoint tensor)."""
    fs = FockSpace(3)
    mb = full_multiplet_basis(fs)
    for n_elec, two_s, dim in mb.sectors:
        assert dim == weyl_paldus(3, n_elec, two_s)
    assert sum(d * (s + 1) for _, s, d in mb.sectors) == fs.dim
    fs2 = FockSpace(2)
    assert [(n, s, d) for n, s, d in full_multiplet_basis(fs2).sectors] == \
        [(0, 0, 1), (1, 1, 2), (2, 0, 3), (2, 2, 1), (3, 1, 2), (4, 0, 1)]
    assert weyl_paldus(6, 6, 0) == 175
    # states are orthonormal multiplets
    for (isec, m), st in mb.states.items():
        assert np.abs(st.T @ st - np.eye(st.shape[1])).max() < 1e-12
    # C1.8: <j'||T~||j> = (-1)^(j-j'+k) sqrt((2j+1)/(2j'+1)) <j||T||j'>
    for op in (fs.t_cd(1), couple(fs.t_cd(0), fs.t_cd(2), 2), couple(fs.t_cd(0), fs.t_ct(1), 2),
               couple(fs.t_cd(2), fs.t_ct(1), 0)):
        red = reduce_tensor(op, mb)
        radj = reduce_tensor(op.adjoint_tensor(), mb)
        assert len(red) == len(radj) > 0
        for (io, ii), r in red.items():
            j, jp = mb.sectors[io][1], mb.sectors[ii][1]
            ph = (-1) ** ((j - jp + op.two_k) // 2) * sqrt((j + 1) / (jp + 1))
            assert np.abs(radj[(ii, io)] - ph * r.T).max() < 1e-12
