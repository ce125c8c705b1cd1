"""GPU parity of the two-pass route of H_eff*Psi (plan flag SU2_PLAN_TWO_PASS, csrc/heff_two_pass.cu) against the
oracle: every element, on workloads whose blocks are ragged against the 64 x 128 tiles, with scratch and chunk sizes
small enough that tasks are cut into several slices, groups and partial slabs."""
import numpy as np
import pytest

from gen.workloads import config_problem, random_psi, synthetic_problem
from helpers import oracle_flat

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _operator(prob, **kw):
    from paper_2309_16724_b200.runtime import HeffOperator
    return HeffOperator(prob, **kw)


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.parametrize("name,scratch,chunk_k", [("mini", 0, 0), ("mini", 4096, 8), ("midi", 0, 0), ("midi", 16384, 24)])
def test_all_tasks_on_the_two_pass_route(name, scratch, chunk_k):
    """min_dim = 1: every task leaves the fused kernel (adjoint, identity, folded and shared operands, alpha per position);
    a scratch of a few KB cuts the tasks into many slices and groups, a short chunk into many partial slabs."""
    torch = _torch()
    prob = config_problem(name)
    op = _operator(prob, large_tiles=True, two_pass=True, two_pass_min_dim=1, two_pass_scratch_bytes=scratch, two_pass_chunk_k=chunk_k)
    assert op.info["two_pass_tasks"] == op.info["ntasks"] and op.info["two_pass_groups"] >= 1
    if scratch:
        assert op.info["two_pass_groups"] > 3
    x = random_psi(op.psi_len, seed=1)
    xd = torch.from_numpy(x).cuda()
    f1 = op.apply(xd).clone()
    f_ref = oracle_flat(prob, op.plan, x)
    assert _rel(f1.cpu().numpy(), f_ref) <= TOL
    assert torch.equal(op.apply(xd), f1)              # deterministic: fixed slab order, no atomics


@pytest.mark.parametrize("min_dim", [1, 40])
def test_hybrid_plan_ragged_tiles(min_dim):
    """L=16, D=500 (block dims 6..109: ragged against 64 x 128 tiles in rows and columns).  min_dim = 40 splits the task list
    between the fused kernel and the two-pass route; both write the same output sectors."""
    torch = _torch()
    prob = synthetic_problem(16, 16, 0, 500, seed=3)
    op = _operator(prob, two_pass=True, two_pass_min_dim=min_dim, two_pass_scratch_bytes=1 << 20, two_pass_chunk_k=256)
    if min_dim > 1:
        assert 0 < op.info["two_pass_tasks"] < op.info["ntasks"]
    x = random_psi(op.psi_len, seed=2)
    f_gpu = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_ref = oracle_flat(prob, op.plan, x)
    assert _rel(f_gpu, f_ref) <= TOL
    # against the fused kernel's result of the same operator
    f_fused = _operator(prob, fused=True).apply(torch.from_numpy(x).cuda()).cpu().numpy()
    assert _rel(f_gpu, f_fused) <= 1e-12


def test_wide_sector_and_both_product_orders():
    """600-wide right sector against 37 / 9-row left sectors: several column tiles, and tasks for which E D^T first is the
    cheaper order (order 1) next to tasks that form A E first."""
    torch = _torch()
    from test_gpu_parity import _wide_problem
    prob = _wide_problem()
    op = _operator(prob, two_pass=True, two_pass_min_dim=1, two_pass_chunk_k=600)
    x = random_psi(op.psi_len, seed=8)
    f_gpu = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_ref = oracle_flat(prob, op.plan, x)
    assert np.abs(f_ref).max() > 0
    assert _rel(f_gpu, f_ref) <= TOL


def test_davidson_and_host_entry_on_a_two_pass_plan():
    torch = _torch()
    prob = config_problem("midi")
    op = _operator(prob, large_tiles=True, two_pass=True, two_pass_min_dim=1)
    ref = _operator(prob)
    x = torch.from_numpy(random_psi(op.psi_len, seed=4)).cuda()
    xh = x.cpu().pin_memory()
    fh = torch.empty_like(xh).pin_memory()
    op.apply_host(xh, fh)
    assert torch.equal(fh, op.apply(x).cpu())
    s1, s2 = op.davidson(x, max_subspace=8), ref.davidson(x, max_subspace=8)
    for _ in range(6):
        t1, r1 = s1.step()
        t2, r2 = s2.step()
        assert abs(t1 - t2) <= 1e-10 * max(1.0, abs(t2)) and abs(r1 - r2) <= 1e-8 * max(1.0, r2)
    s1.close(); s2.close()


def test_caller_owned_scratch_gives_the_same_bits():
    """su2_plan_options.two_pass_scratch_dev: the scratch as a torch tensor (PyTorch owns the memory) instead of an allocation
    of the library's own -- same grouping for the same size, hence the same bits; a buffer that cannot hold one position of
    the largest task is refused."""
    torch = _torch()
    from paper_2309_16724_b200 import Su2Error
    prob = synthetic_problem(16, 16, 0, 500, seed=3)
    nbytes = 1 << 20
    own = _operator(prob, two_pass_scratch_bytes=nbytes, two_pass_chunk_k=256, two_pass_scratch="library")
    ext = _operator(prob, two_pass_scratch_bytes=nbytes, two_pass_chunk_k=256)          # the runtime's default: a torch tensor
    assert own.two_pass_scratch is None and ext.two_pass_scratch is not None and ext.two_pass_scratch.numel() == ext.info["two_pass_scratch_bytes"]
    assert ext.info["two_pass_groups"] == own.info["two_pass_groups"] > 1
    assert ext.info["plan_device_bytes"] < own.info["plan_device_bytes"]
    x = torch.from_numpy(random_psi(own.psi_len, seed=6)).cuda()
    ext.two_pass_scratch.fill_(255)                     # NaN bit patterns: only what an apply wrote itself may be read as data
    ext.two_pass_scratch.zero_()                        # ... the library zeroes the buffer once at plan time; do the same after scribbling
    assert torch.equal(ext.apply(x), own.apply(x))
    from paper_2309_16724_b200 import Plan
    small = torch.empty(4096, dtype=torch.uint8, device="cuda")
    with pytest.raises(Su2Error):
        Plan(prob, family_ptrs={k: t.data_ptr() for k, t in own.family_tensors.items()}, ld_align=own.ld_align,
             two_pass_scratch_bytes=4096, two_pass_scratch_ptr=small.data_ptr())
