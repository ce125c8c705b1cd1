"""ORACLE (test infrastructure only; never imported by the product path).

The renormalisation (blocking) step next to the eigensolver ("5-10 % of the run
time", Eq. (6)-(7): the W^(l) / W^(r) look-ups of block x site products): the block l is
enlarged by the site B, l' = l + B, and every block operator is carried over to the new, rotated and truncated basis.

What the fast path computes with the SU(2) factor of Eq. (5)/(9),

    <(S_l s) J || [O_l x O_B]^k' || (S_l' s') J'> = (-1)^(p_B N_l') C^(S_l, s, J | k_l, k_B, k' | S_l', s', J') <S_l||O_l||S_l'> <s||O_B||s'>,

followed by U[q'_out]^T ( . ) U[q'_in], is obtained HERE without any 6j / 9j symbol: the coupled multiplet states
|(a S_l, sigma s) J M> = sum <S_l M_l; s m|J M> |a M_l> (x) |sigma m> are written out as vectors of the joint Fock space
(Jordan-Wigner, the site is the last orbital: a product state is the block's creation string followed by the site's, so
the joint vector is the Kronecker product), rotated by U, and the operator -- a genuine
Jordan-Wigner matrix of the joint space -- is reduced in that basis with the Wigner-Eckart theorem
(oracle/multiplets.reduce_tensor, which checks every (M, q, M') component).

Pins: tests/test_oracle_blocking.py (the coupled states are orthonormal eigenstates of N, S^2, S_z of the joint space;
blocking the complete basis of n orbitals reproduces, up to the orthogonal change of basis it is, the complete
multiplet basis of n + 1 orbitals: same sector table, same spectrum of the block Hamiltonian).
"""
import numpy as np

from .multiplets import SITE_SECTORS, MultipletBasis, site_multiplet_basis
from .fock import FockSpace
from .wigner import cg


def blocked_basis(basis_l, fs_l, rotation=None):
    """Coupled basis of l' = l + site in FockSpace(fs_l.norb + 1).

    Returns (MultipletBasis of the joint space, sectors, channels): sectors = [(N', twoJ, rows)] sorted by (N', twoJ);
    channels[i] = [(isec_l, sigma, row0)] -- the coupled rows of new sector i are the channels (block sector, site
    multiplet) in this order, channel c holding dim(isec_l) rows from row0.  rotation: {new sector index: (rows x D')
    matrix with orthonormal columns} applied on top (the DMRG truncation); sectors without an entry are dropped."""
    fs_site = FockSpace(1)
    site = site_multiplet_basis(fs_site)
    table = {}
    for il, (nl, sl, dl) in enumerate(basis_l.sectors):
        for sg, (ns, ss) in enumerate(SITE_SECTORS):
            for two_j in range(abs(sl - ss), sl + ss + 1, 2):
                table.setdefault((nl + ns, two_j), []).append((il, sg))
    sectors, channels, states = [], [], {}
    for (n_new, two_j) in sorted(table):
        chans, row0 = [], 0
        for il, sg in table[(n_new, two_j)]:
            chans.append((il, sg, row0))
            row0 += basis_l.sectors[il][2]
        isec = len(sectors)
        sectors.append((n_new, two_j, row0))
        channels.append(chans)
        for two_m in range(-two_j, two_j + 1, 2):
            cols = []
            for il, sg, _ in chans:
                sl, ss = basis_l.sectors[il][1], SITE_SECTORS[sg][1]
                acc = 0.0
                for ml in range(-sl, sl + 1, 2):
                    ms = two_m - ml
                    if abs(ms) > ss or (ms + ss) % 2:
                        continue
                    w = cg(sl, ml, ss, ms, two_j, two_m)
                    if w == 0.0:
                        continue
                    # |a M_l> (x) |sigma m>: block string first, site string last (C1.1)
                    joint = np.einsum("ia,j->ija", basis_l.states[(il, ml)], site.states[(sg, ms)][:, 0])
                    acc = acc + w * joint.reshape(fs_l.dim * 4, -1)
                cols.append(acc)
            states[(isec, two_m)] = np.concatenate(cols, axis=1)
    if rotation is not None:
        new_sec, new_states, new_chan = [], {}, []
        for isec, (n_new, two_j, rows) in enumerate(sectors):
            if isec not in rotation or rotation[isec].shape[1] == 0:
                continue
            u = rotation[isec]
            assert u.shape[0] == rows
            k = len(new_sec)
            new_sec.append((n_new, two_j, u.shape[1]))
            new_chan.append(channels[isec])
            for two_m in range(-two_j, two_j + 1, 2):
                new_states[(k, two_m)] = states[(isec, two_m)] @ u
        return MultipletBasis(new_sec, new_states), sectors, channels
    return MultipletBasis(sectors, states), sectors, channels
