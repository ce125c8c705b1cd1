"""Operator families generated directly in device memory (input generation only; no arithmetic
of the method lives here).

configs[3] (L=76, D=4096) keeps 92 GB of operator blocks resident in HBM; they cannot be staged
through host memory, so their N(0, 1/sqrt(dim_in)) entries are drawn on the device with a seeded
torch generator.  The values are INPUTS: the tests read the few rows the
sampled oracle needs back from the device tensors.

Reproducibility across position shards (paper_2309_16724_b200/sharding.py): the stream of one block is seeded per
group of POS_CHUNK consecutive positions of the FULL family, so a rank that holds positions [lo, hi) draws exactly the
values the single-GPU operator holds at those positions (it generates the groups its slice overlaps and keeps the
slice).
"""
import numpy as np

POS_CHUNK = 32


def device_fill(problem):
    """Returns fill(side, family_index, tensor, offs, lds) for paper_2309_16724_b200.runtime.HeffOperator:
    block b of the family lives at tensor[offs[b]:] as [npos][dim(q_out)][lds[b]] (binding.family_layout)."""
    import torch

    gens = {}

    def fill(side, idx, tensor, offs, lds):
        gen = gens.setdefault(tensor.device, torch.Generator(device=tensor.device))
        fam = (problem.fam_l if side == "l" else problem.fam_r)[idx]
        secs = problem.sec_l if side == "l" else problem.sec_r
        pos0 = getattr(fam, "pos0", 0)                   # first position of a position shard inside the full family
        for b, (qo, qi) in enumerate(zip(fam.q_out, fam.q_in)):
            m, k, ld = secs[qo].dim, secs[qi].dim, lds[b]
            view = tensor[offs[b]:offs[b] + fam.npos * m * ld].view(fam.npos, m, ld)
            std = 1.0 / (k ** 0.5)
            npos_full = getattr(fam, "npos_full", pos0 + fam.npos)
            for c in range(pos0 // POS_CHUNK, (pos0 + fam.npos - 1) // POS_CHUNK + 1):
                g0, g1 = c * POS_CHUNK, min((c + 1) * POS_CHUNK, npos_full)        # the group in the full family
                lo, hi = max(pos0, g0), min(pos0 + fam.npos, g1)                   # the part this tensor holds
                gen.manual_seed(((1 if side == "l" else 2) * 1000 + idx) * 1_000_003 + b * 65_537 + c)
                if (lo, hi) == (g0, g1):
                    view[lo - pos0:hi - pos0].normal_(0.0, std, generator=gen)     # whole group: draw in place
                else:
                    tmp = torch.empty(g1 - g0, m, ld, dtype=torch.float64, device=tensor.device)
                    tmp.normal_(0.0, std, generator=gen)
                    view[lo - pos0:hi - pos0].copy_(tmp[lo - g0:hi - g0])
            if fam.name in ("H_l", "H_r") and qo == qi:
                v = view[:, :, :k]
                v.copy_(0.5 * (v + v.transpose(1, 2)))
    return fill


def device_block_rows(problem, family_tensors, family_layouts):
    """block_rows callback of oracle.heff_sampled.heff_sample reading operator rows back from the
    device tensors (family_tensors[(side, index)] = flat tensor, family_layouts[(side, index)] = (offs, lds))."""
    def rows(side, fam_index, blk, idx, transposed):
        import torch
        fam = (problem.fam_l if side == "l" else problem.fam_r)[fam_index]
        secs = problem.sec_l if side == "l" else problem.sec_r
        offs, lds = family_layouts[(side, fam_index)]
        m, k, ld = secs[fam.q_out[blk]].dim, secs[fam.q_in[blk]].dim, lds[blk]
        view = family_tensors[(side, fam_index)][offs[blk]:offs[blk] + fam.npos * m * ld].view(fam.npos, m, ld)[:, :, :k]
        sel = torch.as_tensor(np.asarray(idx), device=view.device)
        if transposed:
            return view.index_select(2, sel).transpose(1, 2).contiguous().cpu().numpy()
        return view.index_select(1, sel).contiguous().cpu().numpy()
    return rows
