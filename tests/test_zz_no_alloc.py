"""su2_heff_apply_noalloc (include/su2_heff.h): H_eff * Psi with the scratch of the segmented reduction in the library's
static device array -- for callers that cannot allocate device memory -- against the existing path (su2_heff_apply with a
caller-owned workspace).  Collected last on purpose (the suite runs with `pytest -x`): passes alone in a fresh process and
after the other tests, whatever they left in the shared array."""
import numpy as np
import pytest

from gen.workloads import config_problem, random_psi

TOL = 1e-10          # the tolerance of the GPU parity tests (north_star)


@pytest.mark.gpu
@pytest.mark.parametrize("large_tiles,fused", [(False, False), (True, True), (True, False)])
def test_noalloc_apply_equals_the_workspace_path_on_two_calls_in_a_row(large_tiles, fused):
    """Two calls in a row with different Psi (the second one finds the first one's partial tiles in the shared scratch),
    then the first input again: each equals su2_heff_apply's result (same kernels, same order of sums: bit for bit, and a
    fortiori within 1e-10), through the small-block kernel, the fused large-tile (bulk-tensor) kernel and the two-pass route,
    with split segments / partial slabs so that the scratch really carries partial results."""
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2309_16724_b200.binding import noalloc_scratch_bytes
    from paper_2309_16724_b200.runtime import HeffOperator
    prob = config_problem("midi")
    op = HeffOperator(prob, force_split=True, large_tiles=large_tiles, fused=fused)
    assert op.info["nsegments"] > op.info["npsi_sec"] or op.info["two_pass_groups"] > 0      # partial tiles / slabs are in use
    assert 0 < op.plan.workspace_bytes - 256 <= noalloc_scratch_bytes() == 64 * 1024 * 1024
    xs = [torch.from_numpy(random_psi(op.psi_len, seed=s)).cuda() for s in (41, 42, 41)]
    ref = [op.apply(x).clone() for x in xs]                                 # existing path, caller-owned workspace
    for x, want in zip(xs, ref):
        got = torch.full((op.psi_len,), float("nan"), dtype=torch.float64, device="cuda")
        op.apply_noalloc(x, got)
        torch.cuda.synchronize()
        assert torch.isfinite(got).all()
        err = float((got - want).abs().max() / want.abs().max())
        assert err <= TOL, err
        assert torch.equal(got, want)
    # and the oracle agrees with both (the existing path's own gate)
    from helpers import oracle_flat
    f_ref = oracle_flat(prob, op.plan, xs[0].cpu().numpy())
    assert np.abs(ref[0].cpu().numpy() - f_ref).max() / np.abs(f_ref).max() <= TOL


@pytest.mark.gpu
def test_noalloc_apply_rejects_plans_beyond_the_static_scratch():
    """A plan whose partial tiles exceed the 64 MiB array (BASELINE.json configs[2]: 281 MB) is refused with a clear error
    before anything is launched; bad pointers are refused too."""
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2309_16724_b200 import Plan, Su2Error
    from paper_2309_16724_b200.binding import load, noalloc_scratch_bytes
    big = Plan(config_problem("cfg3", fill=False), host_only=True)          # the size check comes first: no device data needed
    assert big.workspace_bytes - 256 > noalloc_scratch_bytes()
    x = torch.zeros(big.psi_len, dtype=torch.float64, device="cuda")
    y = torch.zeros_like(x)
    with pytest.raises(Su2Error) as info:
        big.heff_apply_noalloc(x.data_ptr(), y.data_ptr(), torch.cuda.current_stream().cuda_stream)
    assert "status -8" in str(info.value) and "static scratch holds 67108864" in str(info.value)
    assert load().su2_heff_apply_noalloc(big.handle, x.data_ptr(), x.data_ptr(), None) == -1      # out aliases psi
    assert load().su2_heff_apply_noalloc(None, x.data_ptr(), y.data_ptr(), None) == -1
