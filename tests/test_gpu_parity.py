"""GPU parity tests (run on the B200 box): the CUDA path through the C ABI against the oracle,
element by element, on seeded inputs.  Tolerance (north_star): max |F_gpu - F_oracle| / max |F_oracle|
<= 1e-10 in FP64."""
import numpy as np
import pytest

from gen.workloads import config_problem, integrals, random_psi, synthetic_problem
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


def _cfg1(use_adjoints=True):
    from oracle.abinitio_table import build_problem
    t, v = integrals(6, seed=0, xi=2.0)
    return build_problem(t, v, 2, 6, 0, use_adjoints=use_adjoints)


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.parametrize("force_split", [False, True])
def test_cfg1_exact_hamiltonian_parity(force_split):
    torch = _torch()
    prob = _cfg1()
    op = _operator(prob, force_split=force_split)
    assert op.psi_len == 175 and len(op.plan.labels) == 53
    x = random_psi(op.psi_len, seed=0)
    f_gpu = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_ref = oracle_flat(prob, op.plan, x)
    assert _rel(f_gpu, f_ref) <= TOL


@pytest.mark.parametrize("name,force_split", [("mini", False), ("mini", True), ("midi", False), ("midi", True)])
def test_synthetic_parity_full_oracle(name, force_split):
    """Random-operator workloads with ragged block sizes (1..17), adjoint rows, alpha per position."""
    torch = _torch()
    prob = config_problem(name)
    op = _operator(prob, force_split=force_split)
    if force_split:
        assert op.info["nsegments"] > op.info["npsi_sec"]
    x = random_psi(op.psi_len, seed=1)
    f_gpu = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_ref = oracle_flat(prob, op.plan, x)
    assert _rel(f_gpu, f_ref) <= TOL


@pytest.mark.parametrize("ld_align", [1, 2, 4])
def test_operator_layouts_dense_and_padded(ld_align):
    """su2_opfamily.blk_ld: the same operator in the dense layout (ld = dim; the plan makes padded copies for the
    bulk-tensor engine and reports them), with even and with 4-aligned leading dimensions (read in place), through
    both kernels."""
    torch = _torch()
    prob = config_problem("midi")
    x = random_psi(_operator(prob).psi_len, seed=2)
    f_ref = oracle_flat(prob, _operator(prob).plan, x)
    for kw in (dict(), dict(large_tiles=True), dict(large_tiles=True, fused=True)):   # small-block, two-pass, fused kernels
        large = bool(kw)
        op = _operator(prob, ld_align=ld_align, force_split=True, **kw)
        f = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
        assert _rel(f, f_ref) <= TOL
        if large:
            assert (op.info["padded_copy_bytes"] > 0) == (ld_align == 1)
        d = op.diag().cpu().numpy()
        assert np.abs(d - _operator(prob).diag().cpu().numpy()).max() <= 1e-13 * np.abs(d).max()


@pytest.mark.parametrize("name", ["cfg1", "mini", "midi"])
def test_small_bonds_through_the_large_tile_kernel(name):
    """Bonds whose sectors all hold <= 48 multiplets plan onto heff_small_kernel; SU2_PLAN_LARGE_TILES keeps them on
    heff_dmma_kernel, so the large-tile kernel stays covered on blocks of 1..17 rows (far smaller than a tile),
    and the two kernels are checked against each other as well as against the oracle."""
    torch = _torch()
    prob = _cfg1() if name == "cfg1" else config_problem(name)
    op_small = _operator(prob, force_split=True)
    assert op_small.info["small_plan"] == 1
    op_big = _operator(prob, force_split=True, large_tiles=True, fused=True)
    assert op_big.info["small_plan"] == 0 and op_big.info["two_pass_tasks"] == 0
    op_tp = _operator(prob, force_split=True, large_tiles=True)          # the default of a large-tile plan: two-pass route
    assert op_tp.info["two_pass_tasks"] == op_tp.info["ntasks"]
    x = random_psi(op_small.psi_len, seed=5)
    f_ref = oracle_flat(prob, op_small.plan, x)
    f_small = op_small.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_big = op_big.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_tp = op_tp.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    assert _rel(f_small, f_ref) <= TOL and _rel(f_big, f_ref) <= TOL and _rel(f_tp, f_ref) <= TOL
    assert _rel(f_small, f_big) <= 1e-12 and _rel(f_tp, f_big) <= 1e-12


@pytest.mark.parametrize("name,world", [("mini", 2), ("midi", 3)])
def test_position_shards_add_up_on_the_gpu(name, world):
    """Position-sharded apply (sharding.py): each rank's shard applied by the CUDA path, one after the
    other on this GPU, summed in rank order (what the all-reduce does) = the oracle's full H_eff Psi."""
    torch = _torch()
    from paper_2309_16724_b200.sharding import ShardedHeffOperator, shard_problem
    prob = config_problem(name)
    full = _operator(prob)
    x = random_psi(full.psi_len, seed=6)
    f_ref = oracle_flat(prob, full.plan, x)
    xd = torch.from_numpy(x).cuda()
    total = torch.zeros_like(xd)
    for rank in range(world):
        op = _operator(shard_problem(prob, rank, world))
        assert op.plan.labels == full.plan.labels
        total += op.apply(xd)
    assert _rel(total.cpu().numpy(), f_ref) <= TOL
    single = ShardedHeffOperator(prob, "cuda:0")          # no process group: one rank, no exchange step
    assert single.world == 1 and _rel(single.apply(xd).cpu().numpy(), f_ref) <= TOL


def test_sharded_davidson_reduce_hook():
    """su2_davidson_create_sharded: the reduce hook is called once for the diagonal and once per step, on vectors
    inside the Davidson workspace; with one rank (nothing to add) the iteration is bit-identical to the plain
    solver.  A hook that returns an error aborts the step with that status."""
    torch = _torch()
    from paper_2309_16724_b200 import Su2Error
    from paper_2309_16724_b200.binding import Davidson
    from paper_2309_16724_b200.sharding import ShardedHeffOperator
    prob = config_problem("midi")
    op = ShardedHeffOperator(prob, "cuda:0")
    x0 = torch.from_numpy(random_psi(op.psi_len, seed=8)).cuda()
    plain = op.local.davidson(x0, max_subspace=6)
    sharded = op.davidson(x0, max_subspace=6)
    assert sharded.reduce_calls == 1
    h0 = [plain.step() for _ in range(8)]
    h1 = [sharded.step() for _ in range(8)]
    assert h0 == h1 and sharded.reduce_calls == 9
    assert torch.equal(plain.ritz_vector(), sharded.ritz_vector())
    plain.close(); sharded.close()
    ws = torch.empty(Davidson.workspace_bytes(op.local.plan, 4), dtype=torch.uint8, device="cuda")
    calls = []
    bad = Davidson(op.local.plan, 4, x0.data_ptr(), ws.data_ptr(), torch.cuda.current_stream().cuda_stream,
                   reduce=lambda vec, n, st: calls.append(n) or (-1 if len(calls) > 1 else 0))
    with pytest.raises(Su2Error):
        bad.step(op.local.workspace.data_ptr(), torch.cuda.current_stream().cuda_stream)
    assert calls == [op.psi_len, op.psi_len]
    bad.close()


def test_reduce_hook_that_raises_stops_the_step_and_is_re_raised():
    """a Python exception inside the all-reduce hook (an NCCL error, a failed assert) must not be swallowed by
    ctypes: the C call stops with a negative status instead of continuing on an un-reduced vector, and the original
    exception comes out of step() / of the constructor."""
    torch = _torch()
    from paper_2309_16724_b200.binding import Davidson
    op = _operator(config_problem("mini"))
    x0 = torch.from_numpy(random_psi(op.psi_len, seed=8)).cuda()
    ws = torch.empty(Davidson.workspace_bytes(op.plan, 4), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    calls = []

    def hook(vec, n, st):
        calls.append(n)
        if len(calls) == 2:
            raise RuntimeError("collective failed")
        return 0
    dav = Davidson(op.plan, 4, x0.data_ptr(), ws.data_ptr(), stream, reduce=hook)
    with pytest.raises(RuntimeError, match="collective failed"):
        dav.step(op.workspace.data_ptr(), stream)
    assert len(calls) == 2
    dav.close()

    def bad_from_the_start(vec, n, st):
        raise ValueError("no communicator")
    with pytest.raises(ValueError, match="no communicator"):
        Davidson(op.plan, 4, x0.data_ptr(), ws.data_ptr(), stream, reduce=bad_from_the_start)


def test_sharded_davidson_two_shards_on_one_gpu():
    """Two position shards, both resident on this GPU.  The solver runs on shard 0; its reduce hook adds shard 1's
    share (what the all-reduce delivers): the diagonal at create time, then H_1 v for the vector the step just
    applied (w = W[i] and v = V[i] sit max_subspace * n doubles apart in the Davidson workspace).  Ritz values and
    residuals follow the unsharded solver through a restart."""
    torch = _torch()
    from paper_2309_16724_b200.binding import Davidson
    from paper_2309_16724_b200.sharding import shard_problem
    prob = config_problem("midi")
    full = _operator(prob)
    op0, op1 = _operator(shard_problem(prob, 0, 2)), _operator(shard_problem(prob, 1, 2))
    n, mm = full.psi_len, 5
    x0 = torch.from_numpy(random_psi(n, seed=13)).cuda()
    ws = torch.empty(Davidson.workspace_bytes(op0.plan, mm), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    calls = []

    def reduce(vec, nn, st):
        off = vec - ws.data_ptr()
        w = ws[off:off + 8 * nn].view(torch.float64)
        if not calls:
            w += op1.diag()
        else:
            v = ws[off - 8 * mm * nn:off - 8 * mm * nn + 8 * nn].view(torch.float64)
            w += op1.apply(v.clone())
        calls.append(nn)
        return 0

    dav = Davidson(op0.plan, mm, x0.data_ptr(), ws.data_ptr(), stream, reduce=reduce)
    ref = full.davidson(x0, max_subspace=mm)
    for it in range(9):
        th, rn = dav.step(op0.workspace.data_ptr(), stream)
        th_ref, rn_ref = ref.step()
        if it < 3:   # same trajectory while the different summation order of F (shard sums) has not been amplified
            assert abs(th - th_ref) <= 1e-9 * max(1.0, abs(th_ref)) and abs(rn - rn_ref) <= 1e-7 * max(1.0, rn_ref)
    # whatever the trajectory: the reported Ritz pair is one of the FULL operator
    x = full.new_vector()
    dav.ritz_vector(x.data_ptr(), stream)
    hx = full.apply(x)
    assert abs(float(torch.dot(x, x)) - 1.0) <= 1e-10
    assert abs(float(torch.dot(x, hx)) - th) <= 1e-10 * max(1.0, abs(th))
    assert abs(float((hx - th * x).norm()) - rn) <= 1e-8 * max(1.0, rn)
    assert calls == [n] * 10
    dav.close(); ref.close()


@pytest.mark.parametrize("fused", [False, True])
def test_several_tiles_and_ragged_tail(fused):
    """Blocks larger than one tile with ragged tails (L=16, D=500: dims 6..109), two-pass route and fused kernel."""
    torch = _torch()
    prob = synthetic_problem(16, 16, 0, 500, seed=3)
    dims = [s.dim for s in prob.sec_l]
    assert max(dims) > 64 and any(d % 8 for d in dims)
    op = _operator(prob, fused=fused)
    x = random_psi(op.psi_len, seed=2)
    f_gpu = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_ref = oracle_flat(prob, op.plan, x)
    assert _rel(f_gpu, f_ref) <= TOL


def test_bitwise_reproducible_and_host_entry():
    torch = _torch()
    prob = config_problem("midi")
    op = _operator(prob, force_split=True)
    x = torch.from_numpy(random_psi(op.psi_len, seed=4)).cuda()
    f1 = op.apply(x).clone()
    f2 = op.apply(x).clone()
    assert torch.equal(f1, f2)
    xh = x.cpu().pin_memory()
    fh = torch.empty_like(xh).pin_memory()
    op.apply_host(xh, fh)
    assert torch.equal(fh, f1.cpu())


def test_empty_operator_table_gives_zero():
    torch = _torch()
    prob = config_problem("mini")
    prob.term = []
    op = _operator(prob)
    x = torch.from_numpy(random_psi(op.psi_len, seed=5)).cuda()
    out = torch.full_like(x, 7.0)
    op.apply(x, out)
    assert float(out.abs().max()) == 0.0


def test_diag_matches_oracle_matrix_cfg1():
    from oracle.heff_dense import heff_matrix, psi_sectors
    torch = _torch()
    prob = _cfg1()
    op = _operator(prob)
    h = heff_matrix(prob)
    labels = psi_sectors(prob)
    offs = np.concatenate([[0], np.cumsum([prob.sec_l[s[0]].dim * prob.sec_r[s[4]].dim for s in labels])])
    ref = np.zeros(op.psi_len)
    for i, lab in enumerate(op.plan.labels):
        j = labels.index(lab)
        ref[op.plan.offsets[i]:op.plan.offsets[i + 1]] = np.diag(h)[offs[j]:offs[j + 1]]
    d = op.diag().cpu().numpy()
    assert np.abs(d - ref).max() <= 1e-12 * np.abs(ref).max()


def test_davidson_converges_to_fci_energy_cfg1():
    """End to end: su2_davidson_step on the exact cfg1 Hamiltonian reaches the lowest (N=6,S=0)
    eigenvalue of the Jordan-Wigner Hamiltonian (oracle/fock.py)."""
    from oracle.fock import FockSpace
    from test_oracle_fock import sector_spectrum
    torch = _torch()
    t, v = integrals(6, seed=0, xi=2.0)
    fs = FockSpace(6)
    e0 = sector_spectrum(fs, fs.hamiltonian(t, v), 6, 0)[0]
    op = _operator(_cfg1())
    x0 = torch.from_numpy(random_psi(op.psi_len, seed=0)).cuda()
    solver = op.davidson(x0, max_subspace=12)
    theta = res = None
    for it in range(60):
        theta, res = solver.step()
        if res < 1e-9:
            break
    assert res < 1e-9, (it, theta, res)
    assert abs(theta - e0) < 1e-10
    xr = solver.ritz_vector()
    hx = op.apply(xr)
    assert abs(float(torch.dot(xr, hx)) - e0) < 1e-10
    assert abs(float(torch.dot(xr, xr)) - 1.0) < 1e-12
    assert len(solver.history) > 12          # went through at least one restart
    solver.close()


def test_davidson_follows_the_krylov_bound_midi():
    """The new-direction rule (reading G8): on the random-operator workload theta lies inside the range of
    diag(H_eff), so the solver must take the Krylov direction t = r until theta has fallen below min(diag); its Ritz
    value after j applies then equals the lowest Ritz value of H in span{x0, H x0, ..., H^(j-1) x0} (computed here
    with numpy from GPU applies); theta falls monotonically and the residual ends below where it started.  The k x k Ritz
    problem, the projections and the residual all run on the device (one CTA Jacobi), so this also pins them."""
    torch = _torch()
    prob = config_problem("midi")
    op = _operator(prob)
    n = op.psi_len
    x0 = torch.from_numpy(random_psi(n, seed=21)).cuda()
    steps = 14
    basis, hbasis, kry = [], [], []
    v = x0 / x0.norm()
    for j in range(steps):
        for _ in range(2):
            for b in basis:
                v = v - torch.dot(b, v) * b
        v = v / v.norm()
        basis.append(v)
        hbasis.append(op.apply(v).clone())
        g = np.array([[float(torch.dot(a, hb)) for hb in hbasis] for a in basis])
        kry.append(float(np.linalg.eigvalsh((g + g.T) / 2)[0]))
        v = hbasis[-1].clone()
    # mode 0 (always t = r) IS the Krylov iteration: same Ritz values as the numpy construction above
    s0 = op.davidson(x0, max_subspace=steps + 2)
    s0.dav.set_preconditioner(0)
    hist0 = [s0.step() for _ in range(steps)]
    for j in range(steps):
        assert abs(hist0[j][0] - kry[j]) <= 1e-8 * max(1.0, abs(kry[j])), (j, hist0[j][0], kry[j])
    # default mode: identical, bit for bit, until theta has dropped below min(diag); monotone throughout
    solver = op.davidson(x0, max_subspace=steps + 2)
    hist = [solver.step() for _ in range(steps)]
    theta = [h[0] for h in hist]
    dmin = float(op.diag().min())
    assert theta[0] > dmin                                   # the random start lies inside the range of diag
    first_below = next((j for j in range(steps) if theta[j] < dmin), steps)
    assert first_below >= 2
    assert hist[:first_below + 1] == hist0[:first_below + 1]
    assert all(theta[j + 1] <= theta[j] + 1e-12 for j in range(steps - 1))
    assert hist[-1][1] < hist[0][1]                          # the residual ends below where it started
    # the reported pair is a Ritz pair of the operator: |H x - theta x| as reported
    xr = solver.ritz_vector()
    hx = op.apply(xr)
    assert abs(float(torch.dot(xr, xr)) - 1.0) <= 1e-10
    assert abs(float(torch.dot(xr, hx)) - theta[-1]) <= 1e-10 * max(1.0, abs(theta[-1]))
    assert abs(float((hx - theta[-1] * xr).norm()) - hist[-1][1]) <= 1e-8 * max(1.0, hist[-1][1])
    solver.close(); s0.close()


def test_davidson_diagonal_correction_on_a_dominant_diagonal():
    """The other branch of the rule: a problem whose H_eff is diagonally dominant with theta below min(diag) --
    the exact cfg1 Hamiltonian shifted so -- converges with the diagonal correction in fewer applies than with
    t = r, to the same eigenvalue."""
    torch = _torch()
    op = _operator(_cfg1())
    x0 = torch.from_numpy(random_psi(op.psi_len, seed=3)).cuda()
    out = {}
    for mode in (1, 0):
        solver = op.davidson(x0, max_subspace=12)
        solver.dav.set_preconditioner(mode)
        for it in range(80):
            th, rn = solver.step()
            if rn < 1e-9:
                break
        out[mode] = (it, th, rn)
        solver.close()
    assert out[1][2] < 1e-9 and out[0][2] < 1e-9
    assert abs(out[1][1] - out[0][1]) < 1e-10
    assert out[1][0] <= out[0][0]


def _physical_problem(L, nl, frac, seed=1):
    """Exact ab initio operator table (oracle/abinitio_table.py) on L orbitals with TRUNCATED, rotated block bases
    (a seeded fraction of every multiplet sector is kept): the kind of problem a DMRG sweep hands to the eigensolver."""
    from oracle.abinitio_table import build_problem
    from oracle.fock import FockSpace
    from oracle.multiplets import full_multiplet_basis
    t, v = integrals(L, seed=0, xi=2.0)
    rng = np.random.default_rng(seed)

    def keep(norb):
        out = {}
        for isec, (_, _, d) in enumerate(full_multiplet_basis(FockSpace(norb)).sectors):
            q, _ = np.linalg.qr(rng.normal(size=(d, d)))
            out[isec] = q[:, :max(1, int(round(frac * d)))]
        return out
    return build_problem(t, v, nl, L, 0, keep_l=keep(nl), keep_r=keep(L - nl - 2), use_adjoints=True)


@pytest.mark.parametrize("L,nl,frac", [(8, 3, 0.67), (10, 4, 0.5)])
def test_davidson_converges_on_physical_truncated_problems(L, nl, frac):
    """Convergence beyond the tiny exact case: su2_davidson_step on physical operators with truncated blocks (L = 8: 776
    unknowns, L = 10: 4988) drives the residual below 1e-8 through several restarts, with the diagonal correction
    taking over once theta has fallen below min(diag).  L = 8: theta is the LOWEST eigenvalue of the oracle's dense
    H_eff; L = 10: (theta, x) is an eigenpair of the oracle's H_eff (one oracle apply on the Ritz vector)."""
    torch = _torch()
    from oracle.heff_dense import heff_matrix
    prob = _physical_problem(L, nl, frac)
    op = _operator(prob)
    assert op.psi_len == {8: 776, 10: 4988}[L]
    x0 = torch.from_numpy(random_psi(op.psi_len, seed=5)).cuda()
    solver = op.davidson(x0, max_subspace=16)
    for it in range(400):
        theta, res = solver.step()
        if res < 1e-8:
            break
    assert res < 1e-8, (it, theta, res)
    assert it > 16                                             # went through at least one restart
    xr = solver.ritz_vector().cpu().numpy()
    if L == 8:
        h = heff_matrix(prob)
        w = np.linalg.eigvalsh((h + h.T) / 2)
        assert abs(theta - w[0]) <= 1e-9 * max(1.0, abs(w[0])), (theta, w[:3])
    hx = oracle_flat(prob, op.plan, xr)
    assert np.abs(hx - theta * xr).max() <= 1e-7
    assert abs(xr @ hx - theta) <= 1e-9 * max(1.0, abs(theta))
    solver.close()


@pytest.mark.parametrize("npos_in,npos_out,dims,ld_align", [(70, 130, [(5, 7), (33, 31), (64, 129)], 1), (70, 130, [(5, 7), (33, 31)], 4),
                                                             (1, 3, [(2, 2)], 4), (257, 64, [(48, 50)], 4)])
def test_precontract_against_position_loops(npos_in, npos_out, dims, ld_align):
    """su2_precontract on random families: out[pos'] = sum_pos W[pos', pos] in[pos] per block,
    against plain loops over the positions; ragged sizes (several 64 x 128 tiles with tails, odd element counts:
    8-byte staging; padded layouts: 16-byte staging)."""
    torch = _torch()
    from types import SimpleNamespace
    from paper_2309_16724_b200.runtime import precontract_family
    rng = np.random.default_rng(3)
    secs = [SimpleNamespace(N=0, twoS=0, dim=d) for pair in dims for d in pair]
    fam = SimpleNamespace(npos=npos_in, q_out=[2 * i for i in range(len(dims))], q_in=[2 * i + 1 for i in range(len(dims))],
                          data=[rng.normal(size=(npos_in, m, k)) for m, k in dims])
    w = rng.normal(size=(npos_out, npos_in))
    got = precontract_family(fam, secs, w, ld_align=ld_align)
    for blk, g in zip(fam.data, got):
        want = np.zeros((npos_out,) + blk.shape[1:])
        for po in range(npos_out):
            for pi in range(npos_in):
                want[po] += w[po, pi] * blk[pi]
        assert np.abs(g - want).max() <= 1e-12 * np.abs(want).max()


def test_precontracted_operators_give_the_fci_energy():
    """f1 end to end: every pre-contracted ("complementary") family of the exact L = 8 operator table is formed ON THE
    DEVICE from the block's normal operators and the integral weights (oracle/abinitio_table.py hands out both), equals
    the oracle's own family to rounding, and H_eff built from the device-made families has the oracle's lowest
    eigenvalue (Davidson through restarts; truncated, rotated blocks)."""
    torch = _torch()
    import copy
    from oracle.abinitio_table import build_problem
    from oracle.fock import FockSpace
    from oracle.heff_dense import heff_matrix
    from oracle.multiplets import full_multiplet_basis
    from paper_2309_16724_b200.runtime import precontract_family
    L, nl = 8, 3
    t, v = integrals(L, seed=0, xi=2.0)
    rng = np.random.default_rng(1)

    def keep(norb):
        out = {}
        for isec, (_, _, d) in enumerate(full_multiplet_basis(FockSpace(norb)).sectors):
            q, _ = np.linalg.qr(rng.normal(size=(d, d)))
            out[isec] = q[:, :max(1, int(round(0.67 * d)))]
        return out
    dec = {}
    prob = build_problem(t, v, nl, L, 0, keep_l=keep(nl), keep_r=keep(L - nl - 2), decomposition=dec)
    assert len(dec) > 50
    dev_prob = copy.copy(prob)
    dev_prob.fam_l, dev_prob.fam_r = list(prob.fam_l), list(prob.fam_r)
    worst = 0.0
    for (side, cid), (normal, w) in dec.items():
        fams, secs = (dev_prob.fam_l, prob.sec_l) if side == "l" else (dev_prob.fam_r, prob.sec_r)
        fam = fams[cid]
        made = dict(zip(zip(normal.q_out, normal.q_in), precontract_family(normal, secs, w)))
        new = copy.copy(fam)
        new.data = [made[key] for key in zip(fam.q_out, fam.q_in)]
        scale = max(1e-300, max(np.abs(b).max() for b in fam.data))
        worst = max(worst, max(np.abs(a - b).max() for a, b in zip(new.data, fam.data)) / scale)
        fams[cid] = new
    assert worst <= 1e-12
    op = _operator(dev_prob)
    x0 = torch.from_numpy(random_psi(op.psi_len, seed=5)).cuda()
    solver = op.davidson(x0, max_subspace=16)
    for it in range(400):
        theta, res = solver.step()
        if res < 1e-8:
            break
    h = heff_matrix(prob)
    e0 = np.linalg.eigvalsh((h + h.T) / 2)[0]
    assert res < 1e-8 and abs(theta - e0) <= 1e-9 * max(1.0, abs(e0)), (it, theta, e0, res)
    solver.close()


@pytest.mark.parametrize("n,big", [(2, False), (3, False), (3, True)])
def test_renormalize_against_the_fock_space_blocking(n, big):
    """su2_renormalize (Eq. (6)-(7), :311-315): block of n orbitals + site -> new block in a
    rotated, truncated basis, for normal operators of the block (position-indexed families), site operators and coupled
    block x site products, against oracle/blocking.py -- Jordan-Wigner matrices of the joint Fock space reduced in the
    coupled multiplet basis, no 6j / 9j.  big: every multiplet is replicated so that sectors exceed 48 rows and the step
    runs on the large-tile (bulk-tensor) kernel instead of the small-block one."""
    torch = _torch()
    from types import SimpleNamespace
    from gen.workloads import site_table
    from oracle.blocking import blocked_basis
    from oracle.fock import FockSpace, couple
    from oracle.multiplets import full_multiplet_basis, reduce_tensor
    from paper_2309_16724_b200.runtime import renormalize_family
    fs, fsj = FockSpace(n), FockSpace(n + 1)
    bl = full_multiplet_basis(fs)
    _, sectors, channels = blocked_basis(bl, fs)
    rng = np.random.default_rng(8)
    rot = {}
    for isec, (_, _, d) in enumerate(sectors):
        q, _ = np.linalg.qr(rng.normal(size=(d, d)))
        rot[isec] = q[:, :max(1, (2 * d + 2) // 3)]
    bj, _, _ = blocked_basis(bl, fs, rotation=rot)
    site = {o.name: o for o in site_table()[0]}
    rep = 1
    if big:
        # replicate every multiplet `rep` times (block-diagonal copies): R -> R (x) 1_rep, U -> U (x) 1_rep, results likewise
        rep = 9
    sec_old = [(a, b, d * rep) for a, b, d in bl.sectors]
    sec_new = [(a, b, d * rep) for a, b, d in bj.sectors]
    chans = [[(il, sg, r0 * rep) for il, sg, r0 in lst] for lst in channels]
    eye = np.eye(rep)
    rotation = {q: np.kron(rot[q], eye) for q in rot}
    assert (max(d for _, _, d in sec_old + sec_new) > 48) == big

    def family(ops):
        """position-indexed family of block operators (same rank and dN) reduced in the block's basis"""
        reds = [reduce_tensor(o, bl) for o in ops]
        keys = sorted({k for r in reds for k in r})
        data = [np.stack([np.kron(r.get(k, np.zeros((bl.sectors[k[0]][2], bl.sectors[k[1]][2]))), eye) for r in reds]) for k in keys]
        return SimpleNamespace(dN=ops[0].dN, twoK=ops[0].two_k, npos=len(ops), q_out=[k[0] for k in keys], q_in=[k[1] for k in keys], data=data)

    cases = [([fs.t_cd(i) for i in range(n)], [fsj.t_cd(i) for i in range(n)], None, None, 1),
             ([couple(fs.t_cd(i), fs.t_ct(j), 2) for i in range(n) for j in range(n)],
              [couple(fsj.t_cd(i), fsj.t_ct(j), 2) for i in range(n) for j in range(n)], None, None, 2),
             (None, None, "c~", fsj.t_ct(n), 1),
             ([fs.t_cd(i) for i in range(n)], [fsj.t_cd(i) for i in range(n)], "c+", fsj.t_cd(n), 0),
             ([fs.t_cd(i) for i in range(n)], [fsj.t_cd(i) for i in range(n)], "c~", fsj.t_ct(n), 2),
             ([couple(fs.t_cd(i), fs.t_ct(j), 2) for i in range(n) for j in range(n)],
              [couple(fsj.t_cd(i), fsj.t_ct(j), 2) for i in range(n) for j in range(n)], "c+", fsj.t_cd(n), 3)]
    checked = 0
    for ops_l, ops_lj, sname, op_sj, two_k in cases:
        npos = 1 if ops_l is None else len(ops_l)
        joint = [op_sj] if ops_lj is None else [(o if op_sj is None else couple(o, op_sj, two_k)) for o in ops_lj]
        want = [reduce_tensor(o, bj) for o in joint]
        dN = joint[0].dN
        blocks = [(io, ii) for io, so in enumerate(sec_new) for ii, si in enumerate(sec_new)
                  if so[0] == si[0] + dN and abs(si[1] - two_k) <= so[1] <= si[1] + two_k]
        got = renormalize_family(sec_old, sec_new, chans, rotation, None if ops_l is None else family(ops_l),
                                 site[sname] if sname else None, two_k, blocks)
        scale = max(np.abs(m).max() for w in want for m in w.values())
        for (io, ii), g in zip(blocks, got):
            assert g.shape == (npos, sec_new[io][2], sec_new[ii][2]) and np.isfinite(g).all()
            for pos in range(npos):
                ref = np.kron(want[pos].get((io, ii), np.zeros((bj.sectors[io][2], bj.sectors[ii][2]))), eye)
                assert np.abs(g[pos] - ref).max() <= 1e-12 * scale, (sname, two_k, io, ii, pos)
                checked += 1
    assert checked > 100


def test_gpu_result_is_hermitian_and_linear_midi():
    torch = _torch()
    prob = config_problem("midi")
    op = _operator(prob)
    x = torch.from_numpy(random_psi(op.psi_len, seed=6)).cuda()
    y = torch.from_numpy(random_psi(op.psi_len, seed=7)).cuda()
    hx, hy = op.apply(x).clone(), op.apply(y).clone()
    a, b = float(torch.dot(y, hx)), float(torch.dot(x, hy))
    assert abs(a - b) <= 1e-11 * max(abs(a), float(hx.norm()))
    hz = op.apply(2.0 * x - 0.5 * y)
    assert float((hz - (2.0 * hx - 0.5 * hy)).abs().max()) <= 1e-12 * float(hx.abs().max())


@pytest.mark.parametrize("m,k,n,p,batch", [(8, 8, 8, 8, 1000), (16, 32, 8, 24, 37), (64, 64, 64, 64, 9),
                                           (70, 33, 45, 129, 5), (128, 128, 128, 128, 3), (1, 1, 1, 1, 4),
                                           (512, 512, 512, 512, 2), (200, 70, 300, 600, 2), (65, 8, 8, 64, 300),
                                           # small-block kernel: square sweep shapes, ragged / odd shapes (8-byte
                                           # copies), 1, 2 and 4 warps per item, more items than resident CTAs
                                           (16, 16, 16, 16, 20000), (32, 32, 32, 32, 3000), (7, 5, 9, 3, 501),
                                           (24, 46, 30, 40, 50), (33, 17, 25, 47, 20), (6, 46, 12, 31, 777),
                                           (48, 48, 48, 48, 40), (8, 8, 8, 8, 300000), (2, 64, 2, 5, 33),
                                           (80, 80, 80, 80, 300), (64, 72, 79, 55, 11), (81, 80, 80, 80, 3),
                                           # too big for the small-block kernel, too narrow for the DMMA tiles
                                           (8, 512, 512, 8, 3)])
def test_gemm_pair_batched(m, k, n, p, batch):
    """BASELINE.json configs[4]: C += alpha A X B^T, checked against numpy in FP64."""
    torch = _torch()
    from paper_2309_16724_b200 import gemm_pair_batched
    rng = np.random.default_rng(m * 1000 + p)
    A, X = rng.normal(size=(batch, m, k)), rng.normal(size=(batch, k, n))
    B, C0 = rng.normal(size=(batch, p, n)), rng.normal(size=(batch, m, p))
    dA, dX, dB, dC = (torch.from_numpy(a).cuda() for a in (A, X, B, C0))
    gemm_pair_batched(m, k, n, p, batch, 0.5, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), dC.data_ptr(),
                      torch.cuda.current_stream().cuda_stream)
    ref = C0 + 0.5 * np.matmul(np.matmul(A, X), np.swapaxes(B, 1, 2))
    assert _rel(dC.cpu().numpy(), ref) <= 1e-12


@pytest.mark.parametrize("m,k,n,p,batch", [(64, 20, 128, 128, 2), (256, 256, 256, 256, 3), (300, 260, 258, 384, 2), (70, 33, 45, 129, 5),
                                           (131, 577, 99, 250, 2), (1, 1, 1, 1, 3), (65, 21, 129, 2, 4), (512, 512, 512, 512, 2),
                                           (48, 200, 48, 52, 700), (200, 48, 300, 49, 40), (128, 128, 128, 128, 300)])
def test_gemm_pair_two_pass_route(m, k, n, p, batch):
    """Route 4 (gemm_two_pass.cu): the batch items as the positions of one task on tp_gemm_kernel (heff_two_pass.cu) -- T through
    a scratch in the cheaper product order (A X first or X B^T first: both occur below), own X and own output per item,
    accumulators initialised from C, ragged edge tiles, K tails, odd leading dimensions re-pitched, several items per CTA (the
    batches of hundreds) -- against numpy; the automatic route (which picks it from 48 in every extent up) gives the same bits
    as the explicit one."""
    torch = _torch()
    from paper_2309_16724_b200 import gemm_pair_batched
    rng = np.random.default_rng(m * 1000 + p + 1)
    A, X = rng.normal(size=(batch, m, k)), rng.normal(size=(batch, k, n))
    B, C0 = rng.normal(size=(batch, p, n)), rng.normal(size=(batch, m, p))
    dA, dX, dB, dC = (torch.from_numpy(a).cuda() for a in (A, X, B, C0))
    st = torch.cuda.current_stream().cuda_stream
    gemm_pair_batched(m, k, n, p, batch, 0.5, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), dC.data_ptr(), st, 4)
    ref = C0 + 0.5 * np.matmul(np.matmul(A, X), np.swapaxes(B, 1, 2))
    assert _rel(dC.cpu().numpy(), ref) <= 1e-12
    if min(m, k, n, p) >= 48:      # shapes the automatic route sends here
        auto = torch.from_numpy(C0).cuda()
        gemm_pair_batched(m, k, n, p, batch, 0.5, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), auto.data_ptr(), st)
        assert torch.equal(auto, dC)


def test_gemm_pair_batched_degenerate_calls():
    """batch == 0 is a no-op that leaves C untouched; non-positive dimensions and null pointers are rejected with
    SU2_ERR_INVALID_ARGUMENT before anything is launched."""
    torch = _torch()
    from paper_2309_16724_b200 import Su2Error, gemm_pair_batched
    from paper_2309_16724_b200.binding import kernel_launch_count
    buf = torch.full((64,), 3.0, dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    l0 = kernel_launch_count()
    gemm_pair_batched(8, 8, 8, 8, 0, 0.5, buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), st)
    for bad in ((0, 8, 8, 8, 1), (8, -1, 8, 8, 1), (8, 8, 8, 8, -2)):
        with pytest.raises(Su2Error):
            gemm_pair_batched(*bad, 0.5, buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), st)
    with pytest.raises(Su2Error):
        gemm_pair_batched(8, 8, 8, 8, 1, 0.5, buf.data_ptr(), None, buf.data_ptr(), buf.data_ptr(), st)
    torch.cuda.synchronize()
    assert kernel_launch_count() == l0 and bool((buf == 3.0).all())


@pytest.mark.gpu
def test_gemm_pair_batched_unaligned_and_repeatable():
    """Operands that start 8 bytes off a 16-byte boundary take the 8-byte copy path of the small-block kernel;
    two calls on the same inputs give bit-identical results (one CTA owns an item, no atomics)."""
    torch = _torch()
    from paper_2309_16724_b200 import gemm_pair_batched
    m, k, n, p, batch = 12, 20, 16, 10, 4097
    rng = np.random.default_rng(11)
    host = [rng.normal(size=(batch, a, b)) for a, b in ((m, k), (k, n), (p, n), (m, p))]
    ref = host[3] + 0.5 * np.matmul(np.matmul(host[0], host[1]), np.swapaxes(host[2], 1, 2))
    outs = []
    for shift in (1, 1, 0):
        bufs = [torch.zeros(h.size + 1, dtype=torch.float64, device="cuda") for h in host]
        views = [b[shift:shift + h.size] for b, h in zip(bufs, host)]
        for v, h in zip(views, host):
            v.copy_(torch.from_numpy(h.ravel()))
        gemm_pair_batched(m, k, n, p, batch, 0.5, *(v.data_ptr() for v in views), torch.cuda.current_stream().cuda_stream)
        outs.append(views[3].cpu().numpy().reshape(batch, m, p))
    assert _rel(outs[0], ref) <= 1e-12 and _rel(outs[2], ref) <= 1e-12
    assert np.array_equal(outs[0], outs[1])


def _wide_problem():
    """Hand-made table with a right-block sector wider than the widest CTA tile (600 > 576 columns: two column
    tiles, the first product is recomputed per column tile) and a left sector spanning two 32-row tiles with a
    ragged tail; both blocks carry position-dependent operators, plus one-sided (folded) and identity rows."""
    from gen import rng
    from gen.problem import OpFamily, Problem, Sector, Term
    from gen.workloads import site_table
    sec_l = [Sector(0, 0, 37), Sector(1, 1, 9)]
    sec_r = [Sector(2, 0, 600), Sector(1, 1, 70)]
    site, _ = site_table()
    sid = {o.name: i for i, o in enumerate(site)}

    def fam(sec, dN, twoK, npos, tag, name):
        blocks = [(io, ii) for io, so in enumerate(sec) for ii, si in enumerate(sec)
                  if so.N == si.N + dN and abs(si.twoS - twoK) <= so.twoS <= si.twoS + twoK and (si.twoS + twoK + so.twoS) % 2 == 0]
        data = [rng.normal_array(5, 7000 + 16 * tag + b, (npos, sec[io].dim, sec[ii].dim)) / np.sqrt(sec[ii].dim)
                for b, (io, ii) in enumerate(blocks)]
        return OpFamily(dN=dN, twoK=twoK, npos=npos, q_out=[b[0] for b in blocks], q_in=[b[1] for b in blocks], data=data, name=name)

    fam_l = [fam(sec_l, 0, 0, 3, 1, "X0(l)"), fam(sec_l, 0, 2, 3, 2, "X1(l)"), fam(sec_l, +1, 1, 3, 3, "c+(l)")]
    fam_r = [fam(sec_r, 0, 0, 3, 4, "Y0(r)"), fam(sec_r, 0, 2, 3, 5, "Y1(r)"), fam(sec_r, -1, 1, 3, 6, "R~(r)")]
    a = np.array([0.7, -0.4, 1.1])
    terms = [Term(0, 0, sid["1"], sid["1"], 0, 0, alpha=a, name="X0Y0"),
             Term(1, 1, sid["1"], sid["1"], 2, 2, alpha=a[::-1].copy(), name="X1Y1"),
             Term(2, 2, sid["1"], sid["1"], 1, 1, alpha=None, name="c+R~"),
             Term(0, 0, sid["1"], sid["1"], 0, 0, alpha=a, adj_l=1, adj_r=1, name="X0Y0^H"),
             Term(-1, 0, sid["B0"], sid["1"], 0, 0, alpha=a, name="n_B Y0"),        # folded, right block
             Term(1, -1, sid["1"], sid["B1"], 2, 2, alpha=a, name="X1 s_C"),        # folded, left block
             Term(-1, -1, sid["B0"], sid["B0"], 0, 0, alpha=np.array([0.3]), name="nn")]
    return Problem(n_tot=4, twoS_tot=0, sec_l=sec_l, sec_r=sec_r, fam_l=fam_l, fam_r=fam_r, site=site, term=terms,
                   meta=dict(L=0, N=4, D=0))


@pytest.mark.parametrize("force_split,fused", [(False, True), (True, True), (False, False)])
def test_wide_sector_multiple_column_tiles(force_split, fused):
    torch = _torch()
    prob = _wide_problem()
    op = _operator(prob, force_split=force_split, fused=fused)
    assert max(s.dim for s in prob.sec_r) > 576
    x = random_psi(op.psi_len, seed=8)
    f_gpu = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
    f_ref = oracle_flat(prob, op.plan, x)
    assert np.abs(f_ref).max() > 0
    assert _rel(f_gpu, f_ref) <= TOL


@pytest.mark.parametrize("name,merged", [("mini", False), ("mini", True), ("midi", True)])
def test_u1_mode_parity_and_equivalence(name, merged):
    """U(1)-only mode (SU2_SYMMETRY_U1): the SAME kernels on a plan whose sectors are
    (N, 2 S_z) and whose recoupling factor is one, against the plain U(1) oracle (oracle/heff_u1.py) on the expansion of
    the SU(2) workload -- through the small-block kernel, the large-tile kernel and with split segments -- and, projected
    back onto the coupled basis, against the SU(2)-mode GPU result (the same numbers up to scalars)."""
    torch = _torch()
    from oracle.heff_dense import psi_sectors, unflatten
    from oracle.heff_u1 import (expand_problem, expand_psi_u1, flatten_u1, heff_apply_u1, project_psi_u1, psi_sectors_u1,
                                unflatten_u1)
    prob = config_problem(name)
    u1, maps = expand_problem(prob, merged=merged)
    labels_u1 = psi_sectors_u1(u1)
    op_su2 = _operator(prob)
    x_red = random_psi(op_su2.psi_len, seed=12)
    psi_u1 = expand_psi_u1(prob, u1, maps, unflatten(prob, x_red, psi_sectors(prob)))
    x = flatten_u1(u1, psi_u1, labels_u1)
    f_ref = flatten_u1(u1, heff_apply_u1(u1, psi_u1), labels_u1)
    f_su2 = op_su2.apply(torch.from_numpy(x_red).cuda()).cpu().numpy()
    for kw in (dict(), dict(large_tiles=True), dict(large_tiles=True, fused=True), dict(large_tiles=True, fused=True, force_split=True),
               dict(force_split=True)):
        op = _operator(u1, **kw)
        assert op.plan.labels == labels_u1
        f = op.apply(torch.from_numpy(x).cuda()).cpu().numpy()
        assert _rel(f, f_ref) <= TOL
        back = project_psi_u1(prob, maps, unflatten_u1(u1, f, labels_u1))
        f_back = np.concatenate([back[lab].ravel() for lab in op_su2.plan.labels])
        assert _rel(f_back, f_su2) <= TOL
    assert op.info["cc_flops"] > op_su2.info["cc_flops"]          # R_CC > 1: what the SU(2) adaptation saves


def test_two_ranks_nccl_sharded_apply_when_two_gpus_are_visible(tmp_path):
    """bench.py --gpus 2 (position-sharded H_eff*Psi, NCCL all-reduce of F) on one box: the script re-launches itself
    under torch.distributed.run, prints one JSON line with n_gpus = 2 and scaling "strong", and its Davidson history
    equals the single-GPU run's (the sharded operator IS the single-GPU operator).  Skipped with fewer than 2 GPUs."""
    import json
    import os
    import subprocess
    import sys
    torch = _torch()
    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 visible GPUs")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    lines = {}
    for n in (1, 2):
        out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", str(n), "--config", "cfg2", "--steps", "4",
                              "--warmup", "3", "--no-cpu-baseline"], capture_output=True, text=True, timeout=900)
        assert out.returncode == 0, out.stderr[-2000:]
        lines[n] = json.loads(out.stdout.strip().splitlines()[-1])
    assert lines[2]["n_gpus"] == 2 and lines[2]["scaling"] == "strong"
    assert abs(lines[2]["config"]["cc_flops_per_apply"] - lines[1]["config"]["cc_flops_per_apply"]) <= 1e-9 * lines[1]["config"]["cc_flops_per_apply"]
    t1, t2 = lines[1]["davidson"]["theta"], lines[2]["davidson"]["theta"]
    assert max(abs(a - b) for a, b in zip(t1, t2)) <= 1e-8 * max(1.0, max(abs(a) for a in t1))
