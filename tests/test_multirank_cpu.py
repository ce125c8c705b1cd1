"""N > 1 path on CPU: world_size-2 gloo.  The path shards by replicas only: every
rank plans the same problem and applies its own H_eff; the only cross-rank step is the max-over-ranks
timing reduction of bench.py.  Checked here: identical plans on all ranks (the planner is deterministic),
the MAX reduction, and the whole-job aggregate."""
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
    ms = bench.reduce_max([10.0 + rank, 5.0 - rank], "cpu", world)
    if rank == 0:
        out.put((same, ms, bench.whole_job_tflops(2.0e12, world, ms[0])))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
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
    assert abs(value - 2 * 2.0e12 / 11.0e-3 / 1e12) < 1e-9
