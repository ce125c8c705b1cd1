"""ORACLE (test infrastructure only; never imported by the product path).

SU(2) multiplet bases of a block's Fock space and Wigner-Eckart reduction of spin tensor
operators to "reduced operators" (Sec. II.B).

Wigner-Eckart convention "B" (C1.4):
    <S M; a| T^k_q |S' M'; a'> = <k q; S' M' | S M> * <S a || T^k || S' a'>.

Pins: tests/test_oracle_fock.py (Weyl-Paldus sector counts P6, site table P4 / C1.6,
consistency of every M-component with the reduced element, adjoint rule C1.8).
"""
import numpy as np

from .wigner import cg

# site multiplets sigma0 = (N=0,S=0), sigma1 = (1,1/2), sigma2 = (2,0)  (C1.2)
SITE_SECTORS = ((0, 0), (1, 1), (2, 0))          # (N, two_S)


class MultipletBasis:
    """sectors: list of (N, two_S, dim); states[(isec, two_M)] = array (fock_dim, dim) whose
    columns are the orthonormal states |a, M> of the multiplets a of that sector."""

    def __init__(self, sectors, states):
        self.sectors = sectors
        self.states = states


def full_multiplet_basis(fs):
    """All multiplets of FockSpace fs: for every (N, S) the highest-weight states are the
    S^2 = S(S+1) eigenvectors inside the (N, M=S) subspace; lower M by the ladder operator
    with Condon-Shortley phases, |a,M-1> = S_-|a,M> / sqrt((S+M)(S-M+1))."""
    s2 = fs.s2().toarray()
    sm = fs.sminus().toarray()
    sectors, states = [], {}
    for n_elec in range(0, 2 * fs.norb + 1):
        for two_s in range(n_elec % 2, min(n_elec, 2 * fs.norb - n_elec) + 1, 2):
            idx = fs.sector_indices(n_elec, two_s)
            if len(idx) == 0:
                continue
            w, v = np.linalg.eigh(s2[np.ix_(idx, idx)])
            sel = np.abs(w - 0.25 * two_s * (two_s + 2)) < 1e-9
            if not sel.any():
                continue
            hw = np.zeros((fs.dim, int(sel.sum())))
            hw[idx, :] = v[:, sel]
            isec = len(sectors)
            sectors.append((n_elec, two_s, hw.shape[1]))
            cur = hw
            for two_m in range(two_s, -two_s - 1, -2):
                states[(isec, two_m)] = cur
                if two_m > -two_s:
                    s, m = two_s / 2.0, two_m / 2.0
                    cur = sm @ cur / np.sqrt((s + m) * (s - m + 1))
    return MultipletBasis(sectors, states)


def site_multiplet_basis(fs1):
    """The fixed site multiplets of C1.2 on a one-orbital FockSpace: sigma0 = |0>,
    sigma1 = (c+_u|0>, c+_d|0>), sigma2 = c+_u c+_d|0>."""
    assert fs1.norb == 1
    vac = np.zeros((4, 1))
    vac[0, 0] = 1.0
    up = fs1.cd(0, 0) @ vac
    dn = fs1.cd(0, 1) @ vac
    both = fs1.cd(0, 0) @ (fs1.cd(0, 1) @ vac)
    sectors = [(0, 0, 1), (1, 1, 1), (2, 0, 1)]
    states = {(0, 0): vac, (1, 1): up, (1, -1): dn, (2, 0): both}
    return MultipletBasis(sectors, states)


def truncate_basis(basis, keep):
    """Keep only a subset of multiplets: keep[isec] = orthonormal (dim, newdim) matrix
    (a rotation/selection inside the sector; the same for every M)."""
    sectors, states = [], {}
    for isec, (n, s2, d) in enumerate(basis.sectors):
        if isec not in keep or keep[isec].shape[1] == 0:
            continue
        new = len(sectors)
        sectors.append((n, s2, keep[isec].shape[1]))
        for two_m in range(-s2, s2 + 1, 2):
            states[(new, two_m)] = basis.states[(isec, two_m)] @ keep[isec]
    return MultipletBasis(sectors, states)


def reduce_tensor(op, basis, tol=1e-11):
    """Reduced matrix elements of TensorOp `op` in `basis` (convention B).

    Returns {(isec_out, isec_in): R (dim_out x dim_in)} for the non-zero blocks, after
    checking that EVERY (M, q, M') component equals <k q; S' M'|S M> * R (i.e. that `op`
    really is a rank-k tensor and the basis really consists of multiplets)."""
    out = {}
    k = op.two_k
    for io, (no, so, do) in enumerate(basis.sectors):
        for ii, (ni, si, di) in enumerate(basis.sectors):
            if no != ni + op.dN or not (abs(si - k) <= so <= si + k) or (si + k + so) % 2:
                continue
            red, best = None, 0.0
            elems = {}
            for mi in range(-si, si + 1, 2):
                for q in range(-k, k + 1, 2):
                    mo = mi + q
                    if abs(mo) > so:
                        continue
                    w = cg(k, q, si, mi, so, mo)
                    blk = basis.states[(io, mo)].T @ (op.comp[q] @ basis.states[(ii, mi)])
                    elems[(mo, q, mi)] = (w, blk)
                    if abs(w) > best:
                        best, red = abs(w), blk / w
            if red is None:
                continue
            for (mo, q, mi), (w, blk) in elems.items():
                if np.abs(blk - w * red).max() > tol * max(1.0, np.abs(red).max()):
                    raise ValueError("operator is not a rank-%g tensor in this basis" % (k / 2))
            if np.abs(red).max() > tol:
                out[(io, ii)] = red
    return out
