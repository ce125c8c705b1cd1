"""include/su2_ozaki.h: the FP64 GEMM pair on the INT8 tensor path against oracle/ozaki.py (the
scheme step by step in NumPy: bit for bit, the integer sums are exact and the FP64 recombination has a fixed order) and
against the plain FP64 definition (within 1e-10 of max|C|, the north-star tolerance, and within the scheme's own bound)."""
import numpy as np
import pytest

from oracle import ozaki

TOL = 1e-10


def _torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _stream(torch):
    return torch.cuda.current_stream().cuda_stream


def _operands(seed, batch, m, k, n, p=None, spread=0.0):
    """seeded N(0,1) operands (BASELINE.json configs[4]); spread > 0 multiplies every row of A and column of X by
    2^(uniform(-spread, spread)) so that the per-line scaling matters."""
    rng = np.random.default_rng(seed)
    A, X = rng.normal(size=(batch, m, k)), rng.normal(size=(batch, k, n))
    if spread:
        A *= np.exp2(rng.uniform(-spread, spread, size=(batch, m, 1)))
        X *= np.exp2(rng.uniform(-spread, spread, size=(batch, 1, n)))
    if p is None:
        return A, X
    return A, X, rng.normal(size=(batch, p, n)), rng.normal(size=(batch, m, p))


@pytest.mark.gpu
@pytest.mark.parametrize("m,k,n,batch,nslices,spread", [
    (48, 32, 64, 3, 7, 0.0),          # one tile, ragged in every direction
    (130, 144, 80, 2, 7, 0.0),        # two row tiles with a tail, contraction 144 = one K tile + 16
    (257, 272, 144, 2, 7, 20.0),      # three row tiles, two column tiles, rows / columns of wildly different magnitude
    (128, 128, 128, 5, 4, 0.0),       # fewer slices (the template parameter)
    (64, 512, 256, 2, 2, 3.0),
    (5, 16, 16, 7, 7, 0.0),
    (70, 33, 45, 3, 7, 0.0),          # nothing a multiple of 16, 4 or 2: padded INT8 copies, element-wise FP64 loads
    (131, 577, 100, 2, 7, 4.0),       # a block of BASELINE.json configs[2] / [3]: 131 rows, contraction 577
    (1, 1, 1, 5, 7, 0.0),
    (9, 130, 7, 2, 3, 0.0),
])
def test_i8_matmul_equals_the_oracle_bit_for_bit(m, k, n, batch, nslices, spread):
    torch = _torch()
    from paper_2309_16724_b200.binding import matmul_batched_i8
    A, X = _operands(m * 7 + n, batch, m, k, n, spread=spread)
    A[0, m // 2, :] = 0.0                                         # a zero row and a zero column: exponent 0, all slices 0
    X[0, :, n // 3] = 0.0
    dA, dX = torch.from_numpy(A).cuda(), torch.from_numpy(X).cuda()
    dC = torch.full((batch, m, n), float("nan"), dtype=torch.float64, device="cuda")
    matmul_batched_i8(m, k, n, batch, dA.data_ptr(), dX.data_ptr(), dC.data_ptr(), _stream(torch), nslices)
    torch.cuda.synchronize()
    got = dC.cpu().numpy()
    for b in range(batch):
        want = ozaki.emulated_matmul(A[b], X[b], nslices)
        assert np.array_equal(got[b], want), (b, np.abs(got[b] - want).max())
        exact = A[b] @ X[b]
        assert (np.abs(got[b] - exact) <= ozaki.error_bound(A[b], X[b], nslices) + 4e-16 * np.abs(A[b]) @ np.abs(X[b])).all()
    assert (got[0, m // 2, :] == 0.0).all() and (got[0, :, n // 3] == 0.0).all()


@pytest.mark.gpu
@pytest.mark.parametrize("m,k,n,p,batch", [(48, 32, 64, 20, 3), (130, 144, 80, 132, 2), (256, 256, 256, 256, 3),
                                           (100, 16, 16, 4, 9), (200, 80, 304, 600, 2),
                                           # ragged in every extent (odd row lengths: element-wise loads and stores)
                                           (70, 33, 45, 129, 5), (7, 5, 9, 3, 11), (131, 577, 99, 250, 2), (1, 1, 1, 1, 4)])
def test_i8_gemm_pair_equals_the_oracle_chain_and_the_fp64_definition(m, k, n, p, batch):
    """C += alpha (A X) B^T: the oracle's emulated product applied twice (alpha a power of two, so that alpha * v is exact
    and the final sum is one rounding on both sides): bit for bit; against the plain FP64 definition: 1e-10 of max|C|."""
    torch = _torch()
    from paper_2309_16724_b200.binding import gemm_pair_batched_i8
    A, X, B, C0 = _operands(m + 3 * p, batch, m, k, n, p)
    alpha = -0.5
    dA, dX, dB, dC = (torch.from_numpy(a).cuda() for a in (A, X, B, C0))
    gemm_pair_batched_i8(m, k, n, p, batch, alpha, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), dC.data_ptr(), _stream(torch))
    torch.cuda.synchronize()
    got = dC.cpu().numpy()
    for b in range(batch):
        T = ozaki.emulated_matmul(A[b], X[b])
        want = C0[b] + alpha * ozaki.emulated_matmul(T, B[b].T)
        assert np.array_equal(got[b], want), (b, np.abs(got[b] - want).max())
    ref = C0 + alpha * np.matmul(np.matmul(A, X), np.swapaxes(B, 1, 2))
    assert np.abs(got - ref).max() / np.abs(ref).max() <= TOL
    assert np.abs(got - ref).max() / np.abs(ref).max() <= 1e-12          # what 49 bits give on N(0,1) operands


@pytest.mark.gpu
def test_i8_gemm_pair_chunks_caller_workspace_and_repeats_bit_for_bit():
    """A caller-owned workspace that holds 2 of 5 items (three chunks, the last one ragged) gives the bits of the
    one-chunk run with the library's own stream-ordered allocation; general alpha; a second call accumulates."""
    torch = _torch()
    from paper_2309_16724_b200.binding import gemm_pair_batched_i8, ozaki_launch_count, ozaki_workspace_bytes
    m, k, n, p, batch = 96, 64, 48, 72, 5
    A, X, B, C0 = _operands(11, batch, m, k, n, p)
    dA, dX, dB = (torch.from_numpy(a).cuda() for a in (A, X, B))
    one = torch.from_numpy(C0).cuda()
    l0 = ozaki_launch_count()
    gemm_pair_batched_i8(m, k, n, p, batch, 0.37, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), one.data_ptr(), _stream(torch))
    assert ozaki_launch_count() - l0 == 5 + 14                    # 2 + 7 + 1 + 1 + 7 + 1 kernels per chunk
    nbytes = ozaki_workspace_bytes(m, k, n, p, 2)
    assert ozaki_workspace_bytes(m, k, n, p, 1) < nbytes < ozaki_workspace_bytes(m, k, n, p, 3)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    chunked = torch.from_numpy(C0).cuda()
    l0 = ozaki_launch_count()
    gemm_pair_batched_i8(m, k, n, p, batch, 0.37, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), chunked.data_ptr(), _stream(torch),
                         0, ws.data_ptr(), nbytes)
    assert ozaki_launch_count() - l0 == 3 * 19
    torch.cuda.synchronize()
    assert torch.equal(one, chunked)
    ref = C0 + 0.37 * np.matmul(np.matmul(A, X), np.swapaxes(B, 1, 2))
    assert np.abs(one.cpu().numpy() - ref).max() / np.abs(ref).max() <= 1e-12
    gemm_pair_batched_i8(m, k, n, p, batch, 0.37, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), chunked.data_ptr(), _stream(torch),
                         0, ws.data_ptr(), nbytes)
    torch.cuda.synchronize()
    ref2 = ref + 0.37 * np.matmul(np.matmul(A, X), np.swapaxes(B, 1, 2))
    assert np.abs(chunked.cpu().numpy() - ref2).max() / np.abs(ref2).max() <= 1e-12


@pytest.mark.gpu
def test_i8_gemm_pair_rejects_what_it_cannot_run():
    torch = _torch()
    from paper_2309_16724_b200 import Su2Error
    from paper_2309_16724_b200.binding import gemm_pair_batched_i8, matmul_batched_i8
    buf = torch.zeros(1 << 16, dtype=torch.float64, device="cuda")
    q, st = buf.data_ptr(), _stream(torch)
    gemm_pair_batched_i8(16, 16, 16, 16, 0, 1.0, q, q, q, q, st)                       # batch 0: no-op
    for bad in [(0, 16, 16, 16), (16, 0, 16, 16), (16, 16, -1, 16), (16, 16, 16, 0)]:
        with pytest.raises(Su2Error):
            gemm_pair_batched_i8(*bad, 1, 1.0, q, q, q, q, st)
    with pytest.raises(Su2Error):
        gemm_pair_batched_i8(16, 16, 16, 16, -1, 1.0, q, q, q, q, st)
    with pytest.raises(Su2Error):
        gemm_pair_batched_i8(16, 16, 16, 16, 1, 1.0, q, None, q, q, st)
    with pytest.raises(Su2Error):
        gemm_pair_batched_i8(16, 16, 16, 16, 1, 1.0, q, q, q, q, st, 8)                # nslices out of range
    with pytest.raises(Su2Error):
        gemm_pair_batched_i8(16, 16, 16, 16, 1, 1.0, q, q + 4, q, q, st)               # operand not 8-byte aligned
    with pytest.raises(Su2Error) as info:
        gemm_pair_batched_i8(16, 16, 16, 16, 1, 1.0, q, q, q, q, st, 0, q, 256)        # workspace below one item
    assert "workspace limit below one item" in str(info.value)
    with pytest.raises(Su2Error):
        matmul_batched_i8(16, 20000, 16, 1, q, q, q, st)                               # 7 * 20000 * 127^2 >= 2^31


@pytest.mark.gpu
def test_i8_gemm_pair_at_microbenchmark_size_on_sampled_entries():
    """512^4 (the largest shape of BASELINE.json configs[4]) in the launch configuration bench.py times: sampled entries
    C_ij = C0_ij + alpha a_i^T X b_j from the plain definition in FP64, 1e-10 of max|C|, and bit-reproducible."""
    torch = _torch()
    from paper_2309_16724_b200.binding import gemm_pair_batched_i8
    m = k = n = p = 512
    batch = 12
    A, X, B, C0 = _operands(512, batch, m, k, n, p)
    dA, dX, dB, dC = (torch.from_numpy(a).cuda() for a in (A, X, B, C0))
    dC2 = dC.clone()
    gemm_pair_batched_i8(m, k, n, p, batch, 0.5, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), dC.data_ptr(), _stream(torch))
    gemm_pair_batched_i8(m, k, n, p, batch, 0.5, dA.data_ptr(), dX.data_ptr(), dB.data_ptr(), dC2.data_ptr(), _stream(torch))
    torch.cuda.synchronize()
    assert torch.equal(dC, dC2)
    got = dC.cpu().numpy()
    rng = np.random.default_rng(5)
    scale = np.sqrt(k * n) * 0.5 * 4                                                   # ~ max |alpha a^T X b| over the samples
    worst = 0.0
    for b in range(batch):
        ii, jj = rng.integers(0, m, 48), rng.integers(0, p, 48)
        ii[:4], jj[:4] = [0, m - 1, 127, 128], [p - 1, 0, 128, 127]                    # tile corners
        want = C0[b, ii, jj] + 0.5 * np.einsum("sk,kn,sn->s", A[b, ii], X[b], B[b, jj])
        worst = max(worst, np.abs(got[b, ii, jj] - want).max())
    assert worst <= TOL * scale, worst


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,large_tiles", [("mini", False), ("midi", False), ("midi", True)])
def test_heff_apply_i8_equals_the_oracle_and_the_fp64_path(cfg, large_tiles):
    """su2_heff_apply_i8: every task of the plan (adjoint operands, identity sides, folded one-sided rows, alpha arrays,
    shared and per-position blocks, ragged sectors) on the INT8 tensor path, against the M-resolved oracle (1e-10, the
    tolerance of the FP64 path) and against su2_heff_apply; bit-reproducible."""
    torch = _torch()
    from gen.workloads import config_problem, random_psi
    from helpers import oracle_flat
    from paper_2309_16724_b200.runtime import HeffOperator
    prob = config_problem(cfg)
    op = HeffOperator(prob, large_tiles=large_tiles)
    x = random_psi(op.psi_len, seed=3)
    dx = torch.from_numpy(x).cuda()
    got = op.apply_i8(dx, workspace_bytes=256 << 20).clone()
    again = op.apply_i8(dx, workspace_bytes=256 << 20)
    torch.cuda.synchronize()
    assert torch.equal(got, again)
    f_ref = oracle_flat(prob, op.plan, x)
    scale = np.abs(f_ref).max()
    assert np.abs(got.cpu().numpy() - f_ref).max() / scale <= TOL
    f64 = op.apply(dx)
    assert float((got - f64).abs().max()) / scale <= 1e-11
    # a workspace that holds only a few positions of a task: chunks over the positions; the per-position terms are the same
    # and they are added in the same order, so the bits are the same
    small = op.apply_i8(dx, workspace_bytes=(2 << 20) if cfg == "midi" else (256 << 10))
    assert torch.equal(small, got)
