"""CPU tests of the host logic behind the C ABI: the library loads without a GPU and exports
every symbol include/su2_heff.h declares; the planner's task table (enumeration, recoupling
coefficients, fermion signs, adjoint phases), walked on the host with numpy, equals the oracle."""
import os
import re

import numpy as np
import pytest

from gen.workloads import config_problem, integrals, random_psi
from helpers import host_walk, oracle_flat

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2309_16724_b200.build import build
    build()
    from paper_2309_16724_b200 import load
    return load()


def test_library_exports_every_declared_symbol(lib):
    import ctypes
    header = open(os.path.join(ROOT, "include", "su2_heff.h")).read()
    declared = set(re.findall(r"\b(su2_[a-z0-9_]+)\s*\(", header))
    assert {"su2_plan_create", "su2_heff_apply", "su2_davidson_step"} <= declared
    for name in declared:
        assert hasattr(lib, name), name
    from paper_2309_16724_b200.binding import EXPORTS
    assert set(EXPORTS) == declared
    assert lib.su2_status_string(0) == b"ok"
    # the measurement aid is a library of its own (include/su2_probe.h), outside the product ABI
    assert not hasattr(lib, "su2_probe_fp64_peak")
    probe_h = open(os.path.join(ROOT, "include", "su2_probe.h")).read()
    probe = ctypes.CDLL(os.path.join(ROOT, "paper_2309_16724_b200", "libsu2probe.so"))
    for name in set(re.findall(r"\b(su2_[a-z0-9_]+)\s*\(", probe_h)):
        assert hasattr(probe, name), name
    # the GEMM pair on the INT8 tensor path is a third library (include/su2_ozaki.h); argument checks run without a GPU
    ozaki_h = open(os.path.join(ROOT, "include", "su2_ozaki.h")).read()
    from paper_2309_16724_b200.binding import load_ozaki, ozaki_workspace_bytes
    oz = load_ozaki()
    declared_oz = set(re.findall(r"\b(su2_[a-z0-9_]+)\s*\(", ozaki_h))
    assert {"su2_gemm_pair_batched_i8", "su2_matmul_batched_i8", "su2_ozaki_workspace_bytes"} <= declared_oz
    for name in declared_oz:
        assert hasattr(oz, name), name
    assert oz.su2_gemm_pair_batched_i8(16, 24, 16, 16, 1, 1.0, 16, 16, 16, 16, 9, None, 0, None) == -1
    assert b"nslices" in oz.su2_ozaki_last_error()
    assert ozaki_workspace_bytes(70, 33, 45, 129, 1) == ozaki_workspace_bytes(70, 48, 48, 132, 1)      # padded extents
    assert ozaki_workspace_bytes(512, 512, 512, 512, 1) == 14688256 and ozaki_workspace_bytes(512, 512, 512, 512, 1, 9) == 0
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["su2_heff.h", "su2_ozaki.h", "su2_probe.h"]


def _cfg1(use_adjoints):
    from oracle.abinitio_table import build_problem
    t, v = integrals(6, seed=0, xi=2.0)
    return build_problem(t, v, 2, 6, 0, use_adjoints=use_adjoints)


@pytest.mark.parametrize("which", ["cfg1", "cfg1-adjoint", "mini", "mini-split"])
def test_task_table_equals_oracle(lib, which):
    from paper_2309_16724_b200 import Plan
    prob = _cfg1(which.endswith("adjoint")) if which.startswith("cfg1") else config_problem("mini")
    plan = Plan(prob, host_only=True, force_split=which.endswith("split"))
    if which.startswith("cfg1"):
        assert plan.psi_len == 175 and plan.info["npsi_sec"] == 53
    x = random_psi(plan.psi_len, seed=0)
    ref = oracle_flat(prob, plan, x)
    got = host_walk(prob, plan, x)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    assert plan.info["cc_flops"] > 0 and plan.info["ntask_positions"] >= plan.info["ntasks"]


def test_plan_statistics_of_the_baseline_configs(lib):
    """Shapes of BASELINE.json configs[1..3] under the windowed sector rule (G12)."""
    from paper_2309_16724_b200 import Plan
    expect = {"cfg2": (138, 85126, 6, 46), "cfg3": (138, 1208228, 30, 131), "cfg4": (138, 19728348, 69, 547)}
    for name, (nsec, nelem, dmin, dmax) in expect.items():
        prob = config_problem(name, fill=False)
        dims = [s.dim for s in prob.sec_l]
        assert (min(dims), max(dims)) == (dmin, dmax)
        plan = Plan(prob, host_only=True)
        assert plan.info["npsi_sec"] == nsec and plan.psi_len == nelem
        assert plan.info["nwork_items"] > 0


def test_invalid_inputs_are_rejected(lib):
    from paper_2309_16724_b200 import Plan, Su2Error
    prob = config_problem("mini")
    prob.term[8].twoK_R = prob.term[8].twoK_L + 2           # k1 != k2
    with pytest.raises(Su2Error):
        Plan(prob, host_only=True)
    prob = config_problem("mini")
    prob.fam_l[2].q_out[0] = 99                             # sector out of range
    with pytest.raises(Su2Error):
        Plan(prob, host_only=True)
    prob = config_problem("mini")
    a = np.array(prob.term[10].alpha)
    a[0] = np.nan
    prob.term[10].alpha = a
    with pytest.raises(Su2Error):
        Plan(prob, host_only=True)


def test_device_entry_points_fail_loudly_without_device_plan(lib):
    from paper_2309_16724_b200 import Plan, Su2Error
    plan = Plan(config_problem("mini"), host_only=True)
    with pytest.raises(Su2Error):
        plan.heff_apply(1, 2, 0)


def test_cc_count_matches_the_planner(lib):
    """oracle/cc_count.py (the Python count of the paper's CC, used by bench.py's reference arm) against
    su2_plan_info_t: same tasks, same task-positions (one-sided rows folded to one position, reading G13), same flops."""
    from oracle.cc_count import cc_flops
    from paper_2309_16724_b200 import Plan
    for name in ("mini", "midi", "cfg2"):
        prob = config_problem(name, fill=False)
        plan = Plan(prob, host_only=True)
        cc, ntask, ntp = cc_flops(prob)
        assert ntask == plan.info["ntasks"] and ntp == plan.info["ntask_positions"]
        assert cc == plan.info["cc_flops"]


def test_planner_wigner_symbols_equal_exact_arithmetic_up_to_the_spin_cap(lib):
    """the planner's factorial-based 6j / 9j (long double) against oracle/wigner.py (exact rational arithmetic)
    over the whole admitted range (doubled arguments <= 40); arguments beyond the cap give NaN from the exported symbol and
    SU2_ERR_INVALID_RANK from su2_plan_create instead of silently wrong coefficients."""
    import random
    from oracle.wigner import w6j, w9j
    from paper_2309_16724_b200 import Plan, Su2Error
    from paper_2309_16724_b200.binding import wigner_6j, wigner_9j
    rnd = random.Random(3)
    n = 0
    while n < 1500:
        a, b, d, e = (rnd.randrange(0, 41) for _ in range(4))
        cs = [c for c in range(abs(a - b), min(a + b, 40) + 1, 2) if abs(d - e) <= c <= d + e and (c + d + e) % 2 == 0]
        fs = [f for f in range(abs(a - e), min(a + e, 40) + 1, 2) if abs(b - d) <= f <= b + d and (b + d + f) % 2 == 0]
        if not cs or not fs:
            continue
        c, f = rnd.choice(cs), rnd.choice(fs)
        assert abs(wigner_6j(a, b, c, d, e, f) - w6j(a, b, c, d, e, f)) <= 1e-14
        n += 1
    for args in [(1, 1, 0, 1, 1, 0, 0, 0, 0), (1, 1, 2, 1, 1, 2, 2, 2, 0), (4, 3, 5, 2, 1, 3, 4, 2, 4), (2, 1, 3, 1, 1, 2, 1, 2, 1)]:
        assert abs(wigner_9j(*args) - w9j(*args)) <= 1e-14
    assert wigner_6j(1, 1, 1, 1, 1, 1) == 0.0                       # violates a triangle rule
    assert np.isnan(wigner_6j(42, 2, 42, 2, 42, 2)) and np.isnan(wigner_9j(*([42] * 9)))
    prob = config_problem("mini", fill=False)
    prob.sec_l[0].twoS = 42
    with pytest.raises(Su2Error) as info:
        Plan(prob, host_only=True)
    assert "status -3" in str(info.value)


def test_two_pass_route_planning(lib):
    """Host side of the two-pass route (SU2_PLAN_TWO_PASS, the default of large-tile plans): which tasks take it, how the
    scratch cap cuts them into launch groups, what it adds to the workspace, and that bad options are refused."""
    from paper_2309_16724_b200 import Plan, Su2Error
    prob = config_problem("midi")
    small = Plan(prob, host_only=True)                                   # every sector <= 48 multiplets: small-block kernel
    assert small.info["small_plan"] == 1 and small.info["two_pass_tasks"] == 0 and small.info["two_pass_groups"] == 0
    tp = Plan(prob, host_only=True, large_tiles=True)
    assert tp.info["small_plan"] == 0 and tp.info["two_pass_tasks"] == tp.info["ntasks"] and tp.info["two_pass_groups"] == 1
    assert tp.info["cc_flops"] == small.info["cc_flops"] and tp.info["ntask_positions"] == small.info["ntask_positions"]
    assert tp.info["two_pass_scratch_bytes"] > 0 and tp.workspace_bytes % 256 == 0
    fused = Plan(prob, host_only=True, large_tiles=True, fused=True)
    assert fused.info["two_pass_tasks"] == 0 and fused.info["two_pass_scratch_bytes"] == 0 and fused.info["nwork_items"] > 0
    paced = Plan(prob, host_only=True, large_tiles=True, gang_pacing=True)       # pacing is the fused kernel's: implies it
    assert paced.info["two_pass_tasks"] == 0
    # a scratch of 16 KB: many groups, the same tasks, the same CC; never less than one position of the largest task
    cut = Plan(prob, host_only=True, large_tiles=True, two_pass_scratch_bytes=16384, two_pass_chunk_k=24)
    assert cut.info["two_pass_groups"] > 100 and cut.info["two_pass_tasks"] == tp.info["ntasks"]
    assert cut.info["two_pass_scratch_bytes"] >= 16384 and cut.info["cc_flops"] == tp.info["cc_flops"]
    tiny = Plan(prob, host_only=True, large_tiles=True, two_pass_scratch_bytes=8)
    dmax = max(s.dim for s in prob.sec_l + prob.sec_r)
    assert 8 < tiny.info["two_pass_scratch_bytes"] <= 8 * (dmax * (dmax + 3) + 2 * (dmax + 3))
    # hybrid: only tasks whose four extents reach min_dim leave the fused kernel
    hyb = Plan(prob, host_only=True, large_tiles=True, two_pass_min_dim=10)
    assert 0 < hyb.info["two_pass_tasks"] < hyb.info["ntasks"]
    # executed flops: the cheaper product order and narrow edge tiles; never below CC
    assert tp.info["executed_flops"] >= tp.info["cc_flops"]
    with pytest.raises(Su2Error):
        Plan(prob, host_only=True, large_tiles=True, two_pass_min_dim=-1)
    with pytest.raises(Su2Error):
        Plan(prob, host_only=True, large_tiles=True, two_pass_scratch_bytes=-5)


def test_caller_owned_scratch_is_validated(lib):
    from paper_2309_16724_b200 import Plan, Su2Error
    prob = config_problem("midi")
    ok = Plan(prob, host_only=True, large_tiles=True, two_pass_scratch_bytes=1 << 20, two_pass_scratch_ptr=1 << 20)
    assert ok.info["two_pass_tasks"] == ok.info["ntasks"]
    for kw in (dict(two_pass_scratch_bytes=1 << 20, two_pass_scratch_ptr=(1 << 20) + 8),     # not 256-byte aligned
               dict(two_pass_scratch_bytes=0, two_pass_scratch_ptr=1 << 20),                 # size missing
               dict(two_pass_scratch_bytes=64, two_pass_scratch_ptr=1 << 20)):               # smaller than one position of a task
        with pytest.raises(Su2Error) as info:
            Plan(prob, host_only=True, large_tiles=True, **kw)
        assert "status -7" in str(info.value)
