"""Pins of the blocking oracle (oracle/blocking.py, Eq. (6)-(7), :311-315)."""
import numpy as np
import pytest

from gen.workloads import site_table, weyl_paldus
from oracle.blocking import blocked_basis
from oracle.fock import FockSpace, couple
from oracle.multiplets import SITE_SECTORS, full_multiplet_basis, reduce_tensor
from oracle.wigner import c_hat


@pytest.mark.parametrize("n", [1, 2])
def test_coupled_states_are_multiplets_of_the_joint_space(n):
    fs, fsj = FockSpace(n), FockSpace(n + 1)
    bj, sectors, channels = blocked_basis(full_multiplet_basis(fs), fs)
    num, s2, sz = fsj.number().toarray(), fsj.s2().toarray(), fsj.sz().toarray()
    allv = []
    for isec, (nn, two_j, d) in enumerate(sectors):
        assert d == weyl_paldus(n + 1, nn, two_j)                   # complete block: Weyl-Paldus counts of n + 1 orbitals
        for two_m in range(-two_j, two_j + 1, 2):
            v = bj.states[(isec, two_m)]
            assert np.abs(v.T @ v - np.eye(d)).max() < 1e-12
            assert np.abs(num @ v - nn * v).max() < 1e-12
            assert np.abs(sz @ v - 0.5 * two_m * v).max() < 1e-12
            assert np.abs(s2 @ v - 0.25 * two_j * (two_j + 2) * v).max() < 1e-12
            allv.append(v)
    allv = np.concatenate(allv, axis=1)
    assert allv.shape[1] == fsj.dim and np.abs(allv.T @ allv - np.eye(fsj.dim)).max() < 1e-12   # a complete basis


def test_blocked_hamiltonian_has_the_spectrum_of_the_enlarged_block():
    """The block Hamiltonian of 3 orbitals reduced in the basis blocked from 2 orbitals + site has, sector by sector, the
    eigenvalues it has in the directly constructed multiplet basis of 3 orbitals (an orthogonal change of basis)."""
    rng = np.random.default_rng(2)
    n = 2
    t = rng.normal(size=(n + 1, n + 1)); t = (t + t.T) / 2
    v = rng.normal(size=(n + 1,) * 4)
    v = v + v.transpose(1, 0, 2, 3); v = v + v.transpose(0, 1, 3, 2); v = v + v.transpose(2, 3, 0, 1)
    fs, fsj = FockSpace(n), FockSpace(n + 1)
    from oracle.fock import TensorOp
    h = TensorOp(0, 0, {0: fsj.hamiltonian(t, v)})
    bj, sectors, _ = blocked_basis(full_multiplet_basis(fs), fs)
    direct = full_multiplet_basis(fsj)
    red_b, red_d = reduce_tensor(h, bj), reduce_tensor(h, direct)
    for isec, (nn, two_j, d) in enumerate(sectors):
        jsec = [k for k, s in enumerate(direct.sectors) if s[:2] == (nn, two_j)][0]
        wb = np.linalg.eigvalsh(red_b[(isec, isec)]) if (isec, isec) in red_b else np.zeros(d)
        wd = np.linalg.eigvalsh(red_d[(jsec, jsec)]) if (jsec, jsec) in red_d else np.zeros(d)
        assert np.abs(wb - wd).max() < 1e-11


def test_product_formula_with_the_su2_factor_equals_the_fock_space_reduction():
    """Eq. (5)/(9) in the blocking step (Eq. (6): the W^(l) use): for operators O_l on the block, O_B on the
    site and their coupled products, <(S_l s)J||[O_l x O_B]^k||(S_l' s')J'> = (-1)^(p_B N_l') C^ <S_l||O_l||S_l'><s||O_B||s'>
    against the Jordan-Wigner matrices of the joint space, in a ROTATED, TRUNCATED new basis."""
    n = 2
    fs, fsj = FockSpace(n), FockSpace(n + 1)
    bl = full_multiplet_basis(fs)
    _, sectors, channels = blocked_basis(bl, fs)
    rng = np.random.default_rng(4)
    rot = {}
    for isec, (_, _, d) in enumerate(sectors):
        q, _ = np.linalg.qr(rng.normal(size=(d, d)))
        rot[isec] = q[:, :max(1, (2 * d + 2) // 3)]
    bj, _, _ = blocked_basis(bl, fs, rotation=rot)
    site_ops, _ = site_table()
    site = {o.name: o for o in site_ops}
    cases = [(fs.t_cd(0), fsj.t_cd(0), None, None, 1), (fs.t_ct(1), fsj.t_ct(1), None, None, 1),
             (None, None, "c+", fsj.t_cd(n), 1), (None, None, "B1", couple(fsj.t_cd(n), fsj.t_ct(n), 2), 2),
             (fs.t_cd(1), fsj.t_cd(1), "c+", fsj.t_cd(n), 0), (fs.t_cd(0), fsj.t_cd(0), "c+", fsj.t_cd(n), 2),
             (couple(fs.t_cd(0), fs.t_ct(1), 2), couple(fsj.t_cd(0), fsj.t_ct(1), 2), "c~", fsj.t_ct(n), 1),
             (couple(fs.t_cd(0), fs.t_ct(1), 2), couple(fsj.t_cd(0), fsj.t_ct(1), 2), "c~", fsj.t_ct(n), 3)]
    checked = 0
    for op_l, op_l_joint, sname, op_s_joint, two_k in cases:
        joint = op_l_joint if op_s_joint is None else (op_s_joint if op_l_joint is None else couple(op_l_joint, op_s_joint, two_k))
        want = reduce_tensor(joint, bj)
        red_l = None if op_l is None else reduce_tensor(op_l, bl)
        kl = 0 if op_l is None else op_l.two_k
        so = site[sname] if sname else site["1"]
        got = {}
        for io, (no, jo, _) in enumerate(sectors):
            for ii, (ni, ji, _) in enumerate(sectors):
                acc = np.zeros((sectors[io][2], sectors[ii][2]))
                hit = False
                for lo, sgo, r0 in channels[io]:
                    for li, sgi, c0 in channels[ii]:
                        rs = so.r[sgo][sgi]
                        if rs == 0.0:
                            continue
                        blk = (np.eye(bl.sectors[lo][2]) if lo == li else None) if red_l is None else red_l.get((lo, li))
                        if blk is None:
                            continue
                        coef = c_hat(bl.sectors[lo][1], SITE_SECTORS[sgo][1], jo, kl, so.twoK, two_k,
                                     bl.sectors[li][1], SITE_SECTORS[sgi][1], ji)
                        coef *= (-1) ** ((so.dN & 1) * bl.sectors[li][0]) * rs
                        if coef == 0.0:
                            continue
                        acc[r0:r0 + blk.shape[0], c0:c0 + blk.shape[1]] += coef * blk
                        hit = True
                if hit and np.abs(acc).max() > 1e-13:
                    got[(io, ii)] = rot[io].T @ acc @ rot[ii]
        for key in set(want) | set(got):
            a, b = want.get(key), got.get(key)
            if a is None or b is None:
                assert np.abs(a if b is None else b).max() < 1e-11, key
            else:
                assert np.abs(a - b).max() < 1e-11, key
            checked += 1
    assert checked > 40
