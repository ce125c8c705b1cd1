"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(bench.build_operator): sampled output entries of H_eff * Psi against the M-resolved oracle
(oracle/heff_sampled.py), plus properties that hold at any size
(Hermiticity, linearity, bitwise reproducibility).  Tolerance (north_star): 1e-10 relative to max |F|."""
import numpy as np
import pytest

from gen.workloads import random_psi

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _setup(cfg):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import bench
    prob, op = bench.build_operator(cfg, "cuda:0")
    return torch, prob, op


def _sampled_parity(torch, prob, op, labels_idx, nsamp, block_rows, seed):
    from oracle.heff_dense import expand_psi
    from oracle.heff_sampled import heff_sample
    x = random_psi(op.psi_len, seed=seed)
    f = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    fmax = np.abs(f).max()
    psi_red = {}
    for lab, o0, o1 in zip(op.plan.labels, op.plan.offsets[:-1], op.plan.offsets[1:]):
        psi_red[lab] = x[o0:o1].reshape(prob.sec_l[lab[0]].dim, prob.sec_r[lab[4]].dim)
    full = expand_psi(prob, psi_red)
    rng = np.random.default_rng(seed)
    worst = 0.0
    for si in labels_idx:
        lab = op.plan.labels[si]
        m, p = prob.sec_l[lab[0]].dim, prob.sec_r[lab[4]].dim
        # sampled rows/columns always include the first and the last (ragged tile tails)
        ra = np.unique(np.concatenate([[0, m - 1], rng.choice(m, size=nsamp, replace=False)]))
        rb = np.unique(np.concatenate([[0, p - 1], rng.choice(p, size=nsamp, replace=False)]))
        ref = heff_sample(prob, psi_red, lab, ra, rb, block_rows, psi_full=full)
        got = f[op.plan.offsets[si]:op.plan.offsets[si + 1]].reshape(m, p)[np.ix_(ra, rb)]
        worst = max(worst, np.abs(got - ref).max() / fmax)
    return worst, f


def _sector_choice(prob, op, count):
    """Largest, smallest and a few seeded sectors: all three tile classes appear."""
    sizes = [prob.sec_l[s[0]].dim * prob.sec_r[s[4]].dim for s in op.plan.labels]
    order = np.argsort(sizes)
    rng = np.random.default_rng(7)
    pick = {int(order[-1]), int(order[0]), int(order[len(order) // 2])}
    while len(pick) < count:
        pick.add(int(rng.integers(len(sizes))))
    return sorted(pick)


def test_cfg2_small_block_parity_and_properties():
    """BASELINE.json configs[1]: L=20, D=256, blocks 6-46: the small-block kernel (heff_small_kernel, size classes
    24/40/48) in the launch configuration bench.py times: sampled entries of 24 of the 138 sectors against the
    oracle, every sector against the large-tile kernel on the same plan input, and the any-size properties."""
    import os
    from oracle.heff_sampled import numpy_block_rows
    torch, prob, op = _setup("cfg2")
    assert op.psi_len == 85126 and op.info["small_plan"] == 1
    worst, f = _sampled_parity(torch, prob, op, _sector_choice(prob, op, 24), 5, numpy_block_rows(prob), seed=31)
    assert worst <= TOL, worst
    x = torch.from_numpy(random_psi(op.psi_len, seed=31)).cuda()
    y = torch.from_numpy(random_psi(op.psi_len, seed=32)).cuda()
    hx = op.apply(x).clone()
    assert torch.equal(hx.cpu(), torch.from_numpy(f))                      # bitwise reproducible
    os.environ["SU2_HEFF_SMALL"] = "0"
    try:
        _, _, op_big = _setup("cfg2")
    finally:
        del os.environ["SU2_HEFF_SMALL"]
    assert op_big.info["small_plan"] == 0
    hx_big = op_big.apply(x)
    assert float((hx - hx_big).abs().max()) <= 1e-12 * float(hx.abs().max())   # all 85 126 elements, two kernels
    hy = op.apply(y).clone()
    a, b = float(torch.dot(y, hx)), float(torch.dot(x, hy))
    assert abs(a - b) <= 1e-11 * float(hx.norm()) * float(y.norm())          # Hermiticity
    hz = op.apply(2.0 * x - 0.5 * y)
    assert float((hz - (2.0 * hx - 0.5 * hy)).abs().max()) <= 1e-12 * float(hx.abs().max())


def test_cfg3_sampled_parity_and_properties():
    """BASELINE.json configs[2]: L=40, D=1024, blocks 30-131 (all operators built by the numpy generator)."""
    from oracle.heff_sampled import numpy_block_rows
    torch, prob, op = _setup("cfg3")
    assert op.psi_len == 1208228
    worst, f = _sampled_parity(torch, prob, op, _sector_choice(prob, op, 8), 6, numpy_block_rows(prob), seed=11)
    assert worst <= TOL, worst
    # bitwise reproducibility, Hermiticity <y|Hx> = <Hy|x>, linearity
    x = torch.from_numpy(random_psi(op.psi_len, seed=11)).cuda()
    y = torch.from_numpy(random_psi(op.psi_len, seed=12)).cuda()
    hx = op.apply(x).clone()
    assert torch.equal(hx.cpu(), torch.from_numpy(f))
    hy = op.apply(y).clone()
    a, b = float(torch.dot(y, hx)), float(torch.dot(x, hy))
    assert abs(a - b) <= 1e-11 * float(hx.norm()) * float(y.norm())
    hz = op.apply(2.0 * x - 0.5 * y)
    assert float((hz - (2.0 * hx - 0.5 * hy)).abs().max()) <= 1e-12 * float(hx.abs().max())


def test_cfg4_sampled_parity():
    """BASELINE.json configs[3]: L=76, D=4096, blocks 69-547, 92 GB of operators generated on the device."""
    from gen.device_ops import device_block_rows
    torch, prob, op = _setup("cfg4")
    assert op.psi_len == 19728348
    rows = device_block_rows(prob, op.family_tensors, op.family_layouts)
    worst, _ = _sampled_parity(torch, prob, op, _sector_choice(prob, op, 5), 3, rows, seed=21)
    assert worst <= TOL, worst
