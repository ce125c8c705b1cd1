"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(bench.build_operator): H_eff * Psi against the M-resolved oracle, plus properties that hold at any size
(Hermiticity, linearity, bitwise reproducibility).  Tolerance (north_star): 1e-10 relative to max |F|.

Coverage, elements checked against the oracle / elements of F:
  configs[1] (cfg2):  85 126 / 85 126        -- the FULL oracle (oracle/heff_dense.py), every element
  configs[2] (cfg3):  64 entries (8 x 8) in EVERY one of the 138 sectors = 8 832 / 1 208 228, sampled oracle
  cfg4p (cfg4's blocks, 24 positions): 16 entries in 12 sectors; gang pacing bit-equal, INT8 apply within 1e-12
  configs[3] (cfg4):  36 entries (6 x 6) in 40 of the 138 sectors = 1 440 / 19 728 348, sampled oracle; the sectors
                      are stratified over the three tile classes (all of the two rarer classes' extremes, largest /
                      smallest / median of each) and the sampled rows / columns over the first, a middle and the
                      last row tile / column slab of each sector (incl. the ragged tails).
Launch configuration: bench.build_operator = the library's default plan, which for configs[2..3] / cfg4p is the two-pass
route (SU2_PLAN_TWO_PASS: tp_gemm_kernel, 64 x 128 tiles) and for configs[1] the small-block kernel; the fused large-tile
kernel (SU2_PLAN_FUSED) is compared with it at configs[1], configs[2] and cfg4p.
Every sampled entry is evaluated over ALL operator-table rows, input sectors and positions (oracle/heff_sampled.py)."""
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


def _stratified(dim, tile, count, rng):
    """`count` indices of range(dim): the first and the last one (ragged tails), one inside the last tile, one
    inside a middle tile, the rest seeded."""
    pick = {0, dim - 1, max(0, ((dim - 1) // tile) * tile), min(dim - 1, (dim // (2 * tile)) * tile + tile // 2)}
    while len(pick) < min(count, dim):
        pick.add(int(rng.integers(dim)))
    return np.array(sorted(pick)[:count] if len(pick) > count else sorted(pick))


def _sampled_parity(torch, prob, op, labels_idx, nsamp, block_rows, seed):
    """max over the sampled entries of |F_gpu - F_oracle| / max|F_gpu|, the GPU result, and the number of entries."""
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
    worst, checked = 0.0, 0
    for si in labels_idx:
        lab = op.plan.labels[si]
        m, p = prob.sec_l[lab[0]].dim, prob.sec_r[lab[4]].dim
        ra = _stratified(m, 32, nsamp, rng)      # row tiles of the large-tile kernel are 32 rows
        rb = _stratified(p, 48, nsamp, rng)      # a consumer warp owns 48 columns
        ref = heff_sample(prob, psi_red, lab, ra, rb, block_rows, psi_full=full)
        got = f[op.plan.offsets[si]:op.plan.offsets[si + 1]].reshape(m, p)[np.ix_(ra, rb)]
        worst = max(worst, np.abs(got - ref).max() / fmax)
        checked += got.size
    return worst, f, checked


def _properties(torch, op, f_first, seed, herm_tol=1e-11):
    """bitwise reproducibility (two applies), Hermiticity <y|Hx> = <Hy|x>, linearity H(2x - y/2)."""
    x = torch.from_numpy(random_psi(op.psi_len, seed=seed)).cuda()
    y = torch.from_numpy(random_psi(op.psi_len, seed=seed + 1)).cuda()
    hx = op.apply(x).clone()
    assert torch.equal(hx.cpu(), torch.from_numpy(f_first))
    hy = op.apply(y).clone()
    a, b = float(torch.dot(y, hx)), float(torch.dot(x, hy))
    assert abs(a - b) <= herm_tol * float(hx.norm()) * float(y.norm())
    hz = op.apply(2.0 * x - 0.5 * y)
    assert float((hz - (2.0 * hx - 0.5 * hy)).abs().max()) <= 1e-12 * float(hx.abs().max())
    return x, hx


def test_cfg2_full_oracle_parity_and_properties():
    """BASELINE.json configs[1]: L=20, D=256, blocks 6-46: the small-block kernel (heff_small_kernel, size classes
    24/40/48) in the launch configuration bench.py times, EVERY element against the full oracle; the large-tile
    kernel on the same input as well; the any-size properties."""
    from helpers import oracle_flat
    torch, prob, op = _setup("cfg2")
    assert op.psi_len == 85126 and op.info["small_plan"] == 1 and len(op.plan.labels) == 138
    x = random_psi(op.psi_len, seed=31)
    f = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_ref = oracle_flat(prob, op.plan, x)
    assert np.abs(f - f_ref).max() / np.abs(f_ref).max() <= TOL
    xd, hx = _properties(torch, op, f, 31)
    from paper_2309_16724_b200.runtime import HeffOperator
    for kw in (dict(fused=True), dict()):     # all 85 126 elements through the fused large-tile kernel and the two-pass route
        op_big = HeffOperator(prob, device="cuda:0", large_tiles=True, **kw)
        assert op_big.info["small_plan"] == 0 and (op_big.info["two_pass_tasks"] == 0) == bool(kw)
        f_big = op_big.apply(xd).cpu().numpy()
        assert np.abs(f_big - f_ref).max() / np.abs(f_ref).max() <= TOL


def test_cfg3_sampled_parity_every_sector_and_properties():
    """BASELINE.json configs[2]: L=40, D=1024, blocks 30-131 (all operators built by the numpy generator): 8 x 8
    sampled entries in every one of the 138 sectors."""
    from oracle.heff_sampled import numpy_block_rows
    torch, prob, op = _setup("cfg3")
    assert op.psi_len == 1208228 and len(op.plan.labels) == 138 and op.info["padded_copy_bytes"] == 0
    worst, f, checked = _sampled_parity(torch, prob, op, range(138), 8, numpy_block_rows(prob), seed=11)
    assert checked == 138 * 64
    assert worst <= TOL, worst
    assert op.info["two_pass_tasks"] == op.info["ntasks"]
    x, hx = _properties(torch, op, f, 11)
    from paper_2309_16724_b200.runtime import HeffOperator
    fused = HeffOperator(prob, device="cuda:0", fused=True)      # every element: the fused kernel against the two-pass route
    assert fused.info["two_pass_tasks"] == 0
    assert float((fused.apply(x) - hx).abs().max() / hx.abs().max()) <= 1e-12


def _cfg4_sector_choice(prob, op, count):
    """Sectors stratified over the tile classes of the large-tile kernel (class = smallest of 144 / 288 / 576 columns
    that covers the sector; rows decide the number of row tiles): per class the largest, the smallest and the median
    sector by element count, then seeded picks until `count` sectors."""
    dims = [(prob.sec_l[s[0]].dim, prob.sec_r[s[4]].dim) for s in op.plan.labels]
    cls = [0 if p <= 144 else 1 if p <= 288 else 2 for _, p in dims]
    pick = set()
    for c in range(3):
        members = sorted((m * p, i) for i, ((m, p), cc) in enumerate(zip(dims, cls)) if cc == c)
        if members:
            pick |= {members[0][1], members[-1][1], members[len(members) // 2][1]}
    rng = np.random.default_rng(7)
    while len(pick) < count:
        pick.add(int(rng.integers(len(dims))))
    return sorted(pick), cls


def test_cfg4_sampled_parity_and_properties():
    """BASELINE.json configs[3] (the headline configuration): L=76, D=4096, blocks 69-547, 92 GB of operators
    generated on the device: 6 x 6 sampled entries in 40 sectors over all tile classes and row tiles, then bitwise
    reproducibility, Hermiticity and linearity of the GPU result at this size."""
    from gen.device_ops import device_block_rows
    torch, prob, op = _setup("cfg4")
    assert op.psi_len == 19728348 and op.info["padded_copy_bytes"] == 0 and op.info["two_pass_tasks"] == op.info["ntasks"]
    rows = device_block_rows(prob, op.family_tensors, op.family_layouts)
    sectors, cls = _cfg4_sector_choice(prob, op, 40)
    assert len({cls[i] for i in sectors}) == len(set(cls))
    worst, f, checked = _sampled_parity(torch, prob, op, sectors, 6, rows, seed=21)
    assert checked == 40 * 36
    assert worst <= TOL, worst
    _properties(torch, op, f, 21)


def test_cfg4p_fused_kernel_gang_pacing_and_int8_apply_equal_the_default_apply():
    """cfg4p = the blocks of BASELINE.json configs[3] (69-547 multiplets) with 24 positions per family (5.8 GB): sampled
    entries of the default (two-pass) result against the oracle; the fused kernel (SU2_PLAN_FUSED) agrees with it to 1e-12
    of max|F| on every element; the plan flag SU2_PLAN_GANG_PACING (1 908 row tiles in gangs here) gives the bits of the
    fused plan, twice in a row; the same plan executed on the INT8 tensor path (su2_heff_apply_i8) agrees to 1e-12."""
    from gen.device_ops import device_block_rows, device_fill
    from paper_2309_16724_b200.runtime import HeffOperator
    torch, prob, op = _setup("cfg4p")
    assert op.info["gang_slots"] == 0
    rows = device_block_rows(prob, op.family_tensors, op.family_layouts)
    sectors, _ = _cfg4_sector_choice(prob, op, 12)
    worst, f, checked = _sampled_parity(torch, prob, op, sectors, 4, rows, seed=31)
    assert checked == 12 * 16 and worst <= TOL, worst
    x = torch.from_numpy(random_psi(op.psi_len, seed=31)).cuda()
    want = torch.from_numpy(f).cuda()
    f8 = op.apply_i8(x, workspace_bytes=4 << 30)
    assert float((f8 - want).abs().max() / want.abs().max()) <= 1e-12
    del f8
    op._i8_ws = None
    fused = HeffOperator(prob, device="cuda:0", device_fill=device_fill(prob), fused=True)
    assert fused.info["two_pass_tasks"] == 0 and op.info["two_pass_tasks"] == op.info["ntasks"]
    f_fused = fused.apply(x).clone()
    assert float((f_fused - want).abs().max() / want.abs().max()) <= 1e-12
    del fused
    paced = HeffOperator(prob, device="cuda:0", device_fill=device_fill(prob), gang_pacing=True)
    assert paced.info["gang_slots"] > 1000 and paced.info["two_pass_tasks"] == 0
    for _ in range(2):
        assert torch.equal(paced.apply(x), f_fused)
