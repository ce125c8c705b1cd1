"""B200-native hot path of SU(2) spin-adapted two-site DMRG (arXiv:2309.16724): the superblock
product H_eff * Psi inside a Davidson eigensolver, behind the C ABI of include/su2_heff.h."""
from .binding import (Davidson, Plan, Su2Error, family_block_offsets, family_elems,  # noqa: F401
                      gemm_pair_batched, load)
