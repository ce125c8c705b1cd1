"""ORACLE (test infrastructure only; never imported by the product path).

Jordan-Wigner Fock space, the ab initio Hamiltonian of PAPER.md Eq. (1)
in its spin-free form (reading G7 / SURVEY.md 8(c) C3)

    H = sum_ij t_ij E_ij + 1/2 sum_ijkl (ij|kl) X(i,k,l,j),
    E_ij = sum_s c+_is c_js,  X(i,k,l,j) = sum_st c+_is c+_kt c_lt c_js,

spin operators, elementary spin tensor operators and their couplings.

Conventions:
  * orbitals 0..L-1, modes ordered (0u,0d,1u,1d,...); mode 0 is the most significant
    Kronecker factor; c_mode = Z x ... x Z x a x 1 x ...; a product state is the string
    of creation operators in ascending mode order on the vacuum with sign +1.
  * c+_i is a rank-1/2 tensor with components (+1/2: c+_iu, -1/2: c+_id);
    c~_i is rank 1/2 with components (+1/2: -c_id, -1/2: +c_iu).
  * [T x U]^k_q = sum_q1 <k1 q1; k2 q2|k q> T_q1 U_q2 (operator product in that order).

Pins: tests/test_oracle_fock.py (anticommutators, Hubbard dimer closed form, Heisenberg
dimer / 4-ring energies, tensor-operator commutators with S_z, S_+-).
"""
import numpy as np
import scipy.sparse as sp

from .wigner import cg

_A = sp.csr_matrix(np.array([[0.0, 1.0], [0.0, 0.0]]))      # annihilates: |1> -> |0>
_Z = sp.csr_matrix(np.array([[1.0, 0.0], [0.0, -1.0]]))
_I = sp.identity(2, format="csr")


class FockSpace:
    """Fock space of `norb` spatial orbitals (2*norb modes, dimension 4**norb)."""

    def __init__(self, norb):
        self.norb = norb
        self.nmode = 2 * norb
        self.dim = 4 ** norb
        self._ann = [self._mode_annihilator(p) for p in range(self.nmode)]

    def _mode_annihilator(self, p):
        out = sp.identity(1, format="csr")
        for m in range(self.nmode):
            out = sp.kron(out, _Z if m < p else (_A if m == p else _I), format="csr")
        return out

    # --- elementary operators -------------------------------------------------
    def c(self, i, s):
        """annihilator of orbital i, spin s (0 = up, 1 = down)."""
        return self._ann[2 * i + s]

    def cd(self, i, s):
        return self._ann[2 * i + s].T.tocsr()

    def identity(self):
        return sp.identity(self.dim, format="csr")

    def number(self):
        return sum(self.cd(i, s) @ self.c(i, s) for i in range(self.norb) for s in (0, 1))

    def sz(self):
        return 0.5 * sum(self.cd(i, 0) @ self.c(i, 0) - self.cd(i, 1) @ self.c(i, 1) for i in range(self.norb))

    def splus(self):
        return sum(self.cd(i, 0) @ self.c(i, 1) for i in range(self.norb))

    def sminus(self):
        return self.splus().T.tocsr()

    def s2(self):
        sz = self.sz()
        return self.sminus() @ self.splus() + sz @ sz + sz

    def parity(self):
        """Pi = (-1)^N as a diagonal matrix."""
        n = np.rint(self.number().diagonal()).astype(int)
        return sp.diags((-1.0) ** n).tocsr()

    # --- Hamiltonian of Eq. (1) -----------------------------------------------
    def E(self, i, j):
        return self.cd(i, 0) @ self.c(j, 0) + self.cd(i, 1) @ self.c(j, 1)

    def X(self, i, k, l, j):
        out = sp.csr_matrix((self.dim, self.dim))
        for s in (0, 1):
            for t in (0, 1):
                out = out + self.cd(i, s) @ self.cd(k, t) @ self.c(l, t) @ self.c(j, s)
        return out

    def hamiltonian(self, t, v):
        """H = sum t_ij E_ij + 1/2 sum (ij|kl) X(i,k,l,j); v[i,j,k,l] = (ij|kl)."""
        n = self.norb
        h = sp.csr_matrix((self.dim, self.dim))
        for i in range(n):
            for j in range(n):
                if t[i, j] != 0.0:
                    h = h + t[i, j] * self.E(i, j)
        for i in range(n):
            for j in range(n):
                for k in range(n):
                    for l in range(n):
                        if v[i, j, k, l] != 0.0:
                            h = h + 0.5 * v[i, j, k, l] * self.X(i, k, l, j)
        return h

    # --- spin tensor operators ------------------------------------------------
    def t_cd(self, i):
        """c+_i as a rank-1/2 tensor: {two_q: matrix}."""
        return TensorOp(1, +1, {+1: self.cd(i, 0), -1: self.cd(i, 1)})

    def t_ct(self, i):
        """c~_i as a rank-1/2 tensor (C1.3)."""
        return TensorOp(1, -1, {+1: -self.c(i, 1), -1: self.c(i, 0)})

    def t_identity(self):
        return TensorOp(0, 0, {0: self.identity()})

    def sector_indices(self, n_elec, two_m):
        n = np.rint(self.number().diagonal()).astype(int)
        m2 = np.rint(2 * self.sz().diagonal()).astype(int)
        return np.nonzero((n == n_elec) & (m2 == two_m))[0]


class TensorOp:
    """An irreducible spin tensor operator: rank two_k/2, particle-number change dN,
    components comp[two_q] (sparse matrices), two_q = -two_k, -two_k+2, ..., two_k."""

    def __init__(self, two_k, dN, comp):
        self.two_k = two_k
        self.dN = dN
        self.comp = comp

    def scaled(self, a):
        return TensorOp(self.two_k, self.dN, {q: a * m for q, m in self.comp.items()})

    def plus(self, other):
        assert (self.two_k, self.dN) == (other.two_k, other.dN)
        return TensorOp(self.two_k, self.dN, {q: self.comp[q] + other.comp[q] for q in self.comp})

    def adjoint_tensor(self):
        """T~_q = (-1)^(k+q) (T_{-q})^dagger  (C1.3); same rank, dN -> -dN."""
        return TensorOp(self.two_k, -self.dN,
                        {q: (-1) ** ((self.two_k + q) // 2) * self.comp[-q].T.tocsr() for q in self.comp})


def couple(T, U, two_k):
    """[T x U]^k_q = sum_{q1+q2=q} <k1 q1; k2 q2|k q> T_q1 U_q2  (C1.3)."""
    comp = {}
    for q in range(-two_k, two_k + 1, 2):
        acc = None
        for q1 in T.comp:
            q2 = q - q1
            if q2 not in U.comp:
                continue
            w = cg(T.two_k, q1, U.two_k, q2, two_k, q)
            if w == 0.0:
                continue
            term = w * (T.comp[q1] @ U.comp[q2])
            acc = term if acc is None else acc + term
        if acc is None:
            d = next(iter(T.comp.values())).shape[0]
            acc = sp.csr_matrix((d, d))
        comp[q] = acc
    return TensorOp(two_k, T.dN + U.dN, comp)
