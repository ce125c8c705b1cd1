"""Plain data containers for one two-site superblock problem (the paper's operator-table
and sector-tables).  Shared by the oracle, the tests and the Python binding
as INPUT description only: this module holds no arithmetic of the method.

Subsystems in Jordan-Wigner order: l (left block), B (site), C (site), r (right block).
One operator-table row (`Term`) stands for the rank-0 operator

    X = alpha_pos * [[O_l^{k_l} x O_B^{k_B}]^{k1} x [O_C^{k_C} x O_r^{k_r}]^{k2}]^0 ,  k1 = k2,

summed over the positions `pos` of the block operator families it names: the term has
P = max(npos_l, npos_r) positions; a family with npos == P is indexed by pos, a family with
npos == 1 (or the identity, family -1) is the same for every position.
"""
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np


@dataclass
class Sector:
    N: int          # particle number of the block sector
    twoS: int       # doubled spin
    dim: int        # number of multiplets kept


@dataclass
class OpFamily:
    """Block operators of one type: same (dN, k), same non-zero sector blocks, `npos`
    positions (orbital index or index pair).  data[b] has shape [npos, dim(q_out), dim(q_in)]
    (row-major, positions contiguous per block: PAPER.md:58)."""
    dN: int
    twoK: int
    npos: int
    q_out: List[int]
    q_in: List[int]
    data: List[np.ndarray]
    name: str = ""

    @property
    def parity(self):
        return self.dN & 1


@dataclass
class SiteOp:
    """Reduced elements <sigma_out || O || sigma_in> over the site multiplets
    sigma0=(0,0), sigma1=(1,1/2), sigma2=(2,0)."""
    dN: int
    twoK: int
    r: np.ndarray    # 3x3
    name: str = ""

    @property
    def parity(self):
        return self.dN & 1


@dataclass
class Term:
    fam_l: int                 # family index on l, -1 = identity
    fam_r: int                 # family index on r, -1 = identity
    op_B: int                  # site operator index
    op_C: int
    twoK_L: int                # doubled rank k1 of [O_l x O_B]
    twoK_R: int                # doubled rank k2 of [O_C x O_r]; must equal twoK_L
    alpha: Optional[np.ndarray] = None    # one alpha per position, None = 1.0
    adj_l: int = 0             # 1: use the adjoint tensor T~ of the family (blocks read transposed)
    adj_r: int = 0
    name: str = ""


@dataclass
class Problem:
    n_tot: int
    twoS_tot: int
    sec_l: List[Sector]
    sec_r: List[Sector]
    fam_l: List[OpFamily]
    fam_r: List[OpFamily]
    site: List[SiteOp]
    term: List[Term]
    meta: dict = field(default_factory=dict)
    # "su2": reduced blocks, sectors (N, S), 3 site multiplets.  "u1" (U(1)-only mode): sectors
    # (N, 2 S_z) -- Sector.twoS, OpFamily.twoK and SiteOp.twoK then hold 2 S_z / its change, twoS_tot the target 2 S_z,
    # SiteOp.r is 4 x 4 over the site states |0>, |up>, |down>, |up down>, Term.twoK_L / twoK_R are unused.
    symmetry: str = "su2"

    def npos_of(self, t: Term) -> int:
        pl = self.fam_l[t.fam_l].npos if t.fam_l >= 0 else 1
        pr = self.fam_r[t.fam_r].npos if t.fam_r >= 0 else 1
        assert pl == pr or pl == 1 or pr == 1
        return max(pl, pr)
