"""Position-sharded H_eff*Psi over several GPUs.

The sector tasks are independent and only meet in the accumulation into F ("several million of
independent operations"); the operator families are > 99 % of the bytes, Psi is small.  So the POSITIONS of
every operator-table row are cut into `world` contiguous slices: rank r keeps slice r of every position-indexed
family (and of the row's alpha), applies its share into a private F with the unchanged single-GPU kernels, and
one all-reduce (sum, FP64) of F per apply completes the product -- the one real exchange step of the path.  Psi is
replicated; the Psi layout depends on the sector tables only, so it is identical on all ranks.

`shard_problem` is plain data slicing (no arithmetic of the method).  `ShardedHeffOperator.apply` = the local
`su2_heff_apply` followed by `torch.distributed.all_reduce` (NCCL over NVLink/NVSwitch; gloo in the CPU tests of
the slicing).  The paper does this accumulation with host threads and lists device-to-device pooling as future
work.
"""
import copy

import numpy as np


def position_slice(npos, rank, world):
    """Contiguous, balanced slice [lo, hi) of `npos` positions owned by `rank`."""
    return (npos * rank) // world, (npos * (rank + 1)) // world


def shard_problem(problem, rank, world):
    """The part of `problem` rank `rank` of `world` applies.  Summed over ranks the shards give the full operator.

    * a row with P > 1 positions keeps positions position_slice(P, rank, world) (dropped if that is empty); every
      family it indexes by position is sliced the same way -- a family's slice depends only on its npos, so rows
      that share a family (a row and its Hermitian conjugate) stay consistent;
    * a row with a single position (local terms, identity factors) is kept by rank `row index % world` only;
    * families with one position, sector tables and site operators are replicated.
    Family `data` blocks are sliced as views ([lo:hi] of the leading axis); blocks of a family without host data
    (device-generated workloads) are left to the caller's fill function, only `npos` changes."""
    assert 0 <= rank < world
    if world == 1:
        return problem
    shard = copy.copy(problem)

    def slice_fams(fams):
        out = []
        for f in fams:
            lo, hi = position_slice(f.npos, rank, world)
            if f.npos <= 1 or hi <= lo:
                out.append(f)              # replicated (rows that would need an empty slice are dropped below)
                continue
            g = copy.copy(f)
            g.npos = hi - lo
            g.pos0, g.npos_full = lo, f.npos       # where the slice sits in the full family (device-side generators)
            g.data = [None if b is None else np.ascontiguousarray(b[lo:hi]) for b in f.data] if f.data is not None else None
            out.append(g)
        return out

    shard.fam_l = slice_fams(problem.fam_l)
    shard.fam_r = slice_fams(problem.fam_r)
    terms = []
    for i, t in enumerate(problem.term):
        npos = problem.npos_of(t)
        if npos == 1:
            if i % world == rank:
                terms.append(t)
            continue
        lo, hi = position_slice(npos, rank, world)
        if hi <= lo:
            continue
        u = copy.copy(t)
        if t.alpha is not None:
            u.alpha = np.ascontiguousarray(np.asarray(t.alpha)[lo:hi])
        terms.append(u)
    shard.term = terms
    shard.meta = dict(problem.meta, shard=(rank, world))
    return shard


class ShardedHeffOperator:
    """H_eff of one superblock problem spread over the ranks of a torch.distributed process group, one GPU per
    rank.  apply(psi) returns the full H_eff psi on every rank."""

    def __init__(self, problem, device, group=None, device_fill=None, force_split=False):
        import torch.distributed as dist
        from .runtime import HeffOperator
        self.group = group
        live = dist.is_available() and dist.is_initialized()
        self.rank, self.world = (dist.get_rank(group), dist.get_world_size(group)) if live else (0, 1)
        self.local = HeffOperator(shard_problem(problem, self.rank, self.world), device=device,
                                  device_fill=device_fill, force_split=force_split)
        self.psi_len = self.local.psi_len

    @property
    def info(self):
        return self.local.info

    def apply(self, psi, out=None):
        import torch.distributed as dist
        out = self.local.apply(psi, out)
        if self.world > 1:
            dist.all_reduce(out, op=dist.ReduceOp.SUM, group=self.group)   # on the current stream, after the kernels
        return out

    def new_vector(self):
        return self.local.new_vector()

    def apply_host(self, psi_host, out_host):
        """End-to-end entry with HOST buffers (pinned): H2D of Psi, local su2_heff_apply, all-reduce of F, D2H."""
        import torch
        if not hasattr(self, "_xdev"):
            self._xdev, self._ydev = self.local.new_vector(), self.local.new_vector()
        self._xdev.copy_(psi_host, non_blocking=True)
        self.apply(self._xdev, self._ydev)
        out_host.copy_(self._ydev, non_blocking=True)
        torch.cuda.current_stream(self.local.device).synchronize()
        return out_host

    def davidson(self, x0, max_subspace=20):
        """Davidson solver on the sharded operator: su2_davidson_create_sharded with an all-reduce hook (called on
        the diagonal once and on w = H_eff v every step); everything else is replicated on the ranks."""
        return ShardedDavidsonSolver(self, x0, max_subspace)


class ShardedDavidsonSolver:
    def __init__(self, op, x0, max_subspace=20):
        import torch
        import torch.distributed as dist
        from .binding import Davidson
        self.op, local = op, op.local
        self.ws = torch.empty(Davidson.workspace_bytes(local.plan, max_subspace), dtype=torch.uint8, device=local.device)
        self.stream = torch.cuda.current_stream(local.device).cuda_stream
        self.reduce_calls = 0

        def reduce(vec_ptr, n, stream):
            # the vector lives inside self.ws (the Davidson workspace): view it as a tensor, no copy
            off = vec_ptr - self.ws.data_ptr()
            assert 0 <= off and off + 8 * n <= self.ws.numel() and (stream or 0) == self.stream
            view = self.ws[off:off + 8 * n].view(torch.float64)
            if op.world > 1:
                dist.all_reduce(view, op=dist.ReduceOp.SUM, group=op.group)
            self.reduce_calls += 1
            return 0

        self.dav = Davidson(local.plan, max_subspace, x0.data_ptr(), self.ws.data_ptr(), self.stream, reduce=reduce)
        self.history = []

    def step(self):
        theta, res = self.dav.step(self.op.local.workspace.data_ptr(), self.stream)
        self.history.append((theta, res))
        return theta, res

    def ritz_vector(self):
        x = self.op.local.new_vector()
        self.dav.ritz_vector(x.data_ptr(), self.stream)
        return x

    def close(self):
        self.dav.close()
