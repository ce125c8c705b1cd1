"""N > 1 path on CPU: world_size-2 gloo.  The path shards by operator positions: every rank
plans its slice of the same problem, applies it, and one all-reduce of F completes the product; bench.py adds the
max-over-ranks timing reduction and the sum-over-ranks CC.  Checked here: identical plans on all ranks (the planner
is deterministic), the MAX / SUM reductions of bench.py, and the sharded apply against the oracle."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from gen.workloads import config_problem
    from paper_2309_16724_b200 import Plan
    plan = Plan(config_problem("mini"), host_only=True)
    sig = torch.tensor([plan.psi_len, plan.info["ntasks"], plan.info["nwork_items"],
                        int(np.float64(plan.info["cc_flops"]))], dtype=torch.int64)
    gathered = [torch.zeros_like(sig) for _ in range(world)]
    dist.all_gather(gathered, sig)
    same = all(torch.equal(g, gathered[0]) for g in gathered)
    coef = torch.from_numpy(plan.export_tasks()["coef"])
    ref = coef.clone()
    dist.broadcast(ref, src=0)
    same = same and torch.equal(coef, ref)
    ms = bench.reduce_vals([10.0 + rank, 5.0 - rank], "cpu", world, "max")
    cc = bench.reduce_vals([1.0e12 * (rank + 1)], "cpu", world, "sum")[0]        # the shards' CC add up to the job's
    if rank == 0:
        out.put((same, ms, cc / (ms[0] * 1e-3) / 1e12))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_reductions_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    same, ms, value = out.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert same
    assert ms == [11.0, 5.0]                       # max over ranks of (10, 11) and (5, 4)
    assert abs(value - 3.0e12 / 11.0e-3 / 1e12) < 1e-9


# ---- position-sharded apply (paper_2309_16724_b200/sharding.py) ---------------------------
def _shard_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from gen.workloads import config_problem, random_psi
    from helpers import oracle_flat
    from paper_2309_16724_b200 import Plan
    from paper_2309_16724_b200.sharding import shard_problem
    prob = config_problem("mini")
    shard = shard_problem(prob, rank, world)
    plan_full, plan = Plan(prob, host_only=True), Plan(shard, host_only=True)
    same_layout = plan.labels == plan_full.labels and list(plan.offsets) == list(plan_full.offsets)
    x = random_psi(plan.psi_len, seed=3)
    f = torch.from_numpy(oracle_flat(shard, plan, x))        # this rank's share, by the oracle
    dist.all_reduce(f, op=dist.ReduceOp.SUM)                 # the path's one exchange step
    if rank == 0:
        ref = oracle_flat(prob, plan_full, x)
        out.put((same_layout, float(np.abs(f.numpy() - ref).max() / np.abs(ref).max()), len(shard.term), len(prob.term)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_position_sharding_gloo():
    """Sum over ranks of the sharded operators = the full operator (oracle on each shard, gloo all-reduce)."""
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    same_layout, err, nterm_shard, nterm = out.get(timeout=400)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert same_layout
    assert err <= 1e-13
    assert 0 < nterm_shard <= nterm


def test_position_sharding_partitions_every_row():
    """world = 3 and 5 (more ranks than positions for some rows): every (row, position) lands on exactly one
    rank, families and alphas are sliced alike, and the planner's task tables of the shards add up to the full
    H_eff Psi (host walk of the exported tasks)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from gen.workloads import config_problem, random_psi
    from helpers import host_walk
    from paper_2309_16724_b200 import Plan
    from paper_2309_16724_b200.sharding import position_slice, shard_problem
    prob = config_problem("mini")
    plan_full = Plan(prob, host_only=True)
    x = random_psi(plan_full.psi_len, seed=9)
    ref = host_walk(prob, plan_full, x)
    for world in (3, 5):
        total, npos_sum = np.zeros_like(ref), 0
        for rank in range(world):
            shard = shard_problem(prob, rank, world)
            for t in shard.term:
                npos = shard.npos_of(t)
                npos_sum += npos
                assert t.alpha is None or len(t.alpha) == npos
            total += host_walk(shard, Plan(shard, host_only=True), x)
        assert npos_sum == sum(prob.npos_of(t) for t in prob.term)
        assert np.abs(total - ref).max() <= 1e-13 * np.abs(ref).max()
    assert [position_slice(7, r, 3) for r in range(3)] == [(0, 2), (2, 4), (4, 7)]
    assert position_slice(2, 1, 5) == (0, 0)          # empty slice: the row is dropped on that rank
