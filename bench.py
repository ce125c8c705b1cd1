#!/usr/bin/env python
"""bench.py -- effective FP64 TFLOPS of H_eff*Psi (BASELINE.json metric) on N B200 GPUs.

A "step" is one Davidson iteration on the named workload: su2_davidson_step = one full
H_eff*Psi (fused GEMM-pair kernel + deterministic segmented reduction, SURVEY.md 8(a) a4+a5)
followed by the Rayleigh-Ritz / residual / orthogonalisation vector algebra (a6).  The plan
(a1-a3) is built once per bond before the timed region, as in the paper ("execution ... follows
only after such initialization procedure is completed"); its wall time is reported.

value = CC flops of all ranks / max-over-ranks device time, CC = sum over task-positions of
min(2mkn+2mnp, 2knp+2mkp) (the paper's definition of TFLOPS).

N > 1 (launched by the driver under torch.distributed.run, or re-launched that way by this script when it is
started plainly with --gpus N): ONE H_eff*Psi spread over the ranks by operator positions (sharding.py, SURVEY.md
8(e)): local su2_heff_apply + one FP64 all-reduce of F per step; "scaling": "strong".  --parallelism replicas runs
N independent copies instead ("weak").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg4] [--impl reference] [--parallelism shard|replicas]
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

METRIC = "effective FP64 TFLOPS of H_eff*Psi (CC / time)"
UNIT = "TFLOP/s"
# MEASURED_PEAKS.json has no FP64 entry.  Two denominators are reported:
#  * roofline.peak = the FP64 tensor (DMMA.8x8x4) rate measured live by su2_probe_fp64_peak in this very
#    run (37.1 TFLOP/s = 99.8 % of 148 SM x 64 FMA/clk x 2 x 1.965 GHz): the stricter of the two;
#  * roofline.peak_bf16_ratio_rule = measured bf16 peak x the guide's nominal FP64/BF16 ratio
#    (45 / 2250, blackwell_cuda_programming.md "B200's 45"), the rule for a dtype without a measured peak.
FP64_OVER_BF16_NOMINAL = 45.0 / 2250.0


def ncu_traffic(cfg_name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the committed ncu capture
    of this workload with the round's final build (profiles/r02_traffic_per_launch.txt), or None."""
    path = os.path.join(ROOT, "profiles", "r02_traffic_per_launch.txt")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f).get(cfg_name)
    return None


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return d, "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        for ln in self.lines:
            p = [x.strip() for x in ln.split(",")]
            if len(p) < 9:
                continue
            try:
                sm.append(float(p[1])); mx.append(float(p[2])); power.append(float(p[3]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------ CPU oracle arm
# Bounded, seeded, STRATIFIED sample of the operator-table rows (SURVEY.md 8(d) "CPU baseline"): every row (Term) is a
# stratum; of its P positions floor(frac * P + u) are kept (u: one seeded uniform per row, systematic sampling), rows
# that keep none are dropped.  Block sizes, sector tables and Psi are the full workload's.  The sample fraction is
# chosen per config so that one oracle apply takes some seconds on the box's cores; the TFLOP/s figure is intensive,
# the full-apply time quoted next to it is EXTRAPOLATED from it (CC of the full workload / measured rate).
SAMPLE_FRAC = {"cfg1": 1.0, "mini": 1.0, "midi": 1.0, "cfg2": 1.0, "cfg3": 0.01, "cfg4": 0.0002, "cfg4p": 0.02}


def oracle_sample_problem(cfg_name, frac, seed=0):
    import copy
    import numpy as np
    from gen import workloads as W
    from gen.problem import Problem
    c = W.CONFIGS[cfg_name]
    if cfg_name == "cfg1":
        from oracle.abinitio_table import build_problem
        t, v = W.integrals(c["L"], seed=0, xi=c["xi"])
        return build_problem(t, v, 2, c["N"], c["twoS"], use_adjoints=True), "all rows, all positions"
    full = W.synthetic_problem(c["L"], c["N"], c["twoS"], c["D"], xi=c["xi"], seed=0, fill=frac >= 1.0,
                               pos_cap=c.get("pos_cap"))
    if frac >= 1.0:
        return full, "all rows, all positions"
    rng = np.random.default_rng(seed)
    keeps = [int(np.floor(frac * full.npos_of(t) + rng.random())) for t in full.term]
    if not any(keeps):                                       # never an empty sample: one position of the longest row
        keeps[int(np.argmax([full.npos_of(t) for t in full.term]))] = 1
    fam_l, fam_r, terms, kept_rows, kept_pos, tot_pos = [], [], [], 0, 0, 0
    for ti, t in enumerate(full.term):
        npos = full.npos_of(t)
        tot_pos += npos
        keep = keeps[ti]
        if keep <= 0:
            continue
        kept_rows += 1
        kept_pos += keep
        t = copy.copy(t)
        for side, fams, secs, new in (("l", full.fam_l, full.sec_l, fam_l), ("r", full.fam_r, full.sec_r, fam_r)):
            idx = t.fam_l if side == "l" else t.fam_r
            if idx < 0:
                continue
            f = fams[idx]
            nf = W.make_family(secs, f.dN, f.twoK, min(keep, f.npos), 0, 900 + 2 * ti + (side == "r"), f.name,
                               symmetric=f.name in ("H_l", "H_r"))
            new.append(nf)
            if side == "l":
                t.fam_l = len(new) - 1
            else:
                t.fam_r = len(new) - 1
        t.alpha = None if t.alpha is None else np.asarray(t.alpha)[:keep]
        if t.alpha is not None and len(t.alpha) < keep:       # a single-position alpha of a one-position row
            t.alpha = np.resize(t.alpha, keep)
        terms.append(t)
    prob = Problem(n_tot=full.n_tot, twoS_tot=full.twoS_tot, sec_l=full.sec_l, sec_r=full.sec_r, fam_l=fam_l,
                   fam_r=fam_r, site=full.site, term=terms, meta=dict(full.meta))
    what = ("seeded stratified sample: %d of %d operator-table rows, %d of %d row-positions (fraction %.4g per row), "
            "all sector combinations, full block sizes" % (kept_rows, len(full.term), kept_pos, tot_pos, frac))
    return prob, what


def time_oracle(cfg_name, budget_s=20.0, threads=None):
    """Times oracle.heff_dense.heff_apply, as it stands, on the bounded sample.  Nothing of the CUDA library is loaded:
    the Psi layout comes from oracle.heff_dense.psi_sectors, the flop count from oracle.cc_count."""
    import numpy as np
    from gen.workloads import random_psi
    from oracle.cc_count import cc_flops
    from oracle.heff_dense import heff_apply, psi_sectors, unflatten
    from threadpoolctl import threadpool_info, threadpool_limits
    prob, what = oracle_sample_problem(cfg_name, SAMPLE_FRAC.get(cfg_name, 1.0))
    labels = psi_sectors(prob)
    n = sum(prob.sec_l[s[0]].dim * prob.sec_r[s[4]].dim for s in labels)
    psi = unflatten(prob, random_psi(n, seed=0), labels)
    cc, _, _ = cc_flops(prob)

    def run(limit):
        times = []
        with threadpool_limits(limits=limit):
            while True:
                t0 = time.perf_counter()
                heff_apply(prob, psi, check_leak=False)
                times.append(time.perf_counter() - t0)
                if sum(times) > budget_s / 2 or len(times) >= 3:
                    break
        return min(times)
    cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1]) if threads is None else threads
    t_all = run(threads)
    t_one = run(1)
    return {"value": cc / t_all / 1e12, "unit": UNIT, "cores": int(cores), "kind": "oracle",
            "sample": what + "; CC of the sample %.3e flop" % cc, "seconds_per_sample_apply": t_all,
            "single_thread": {"value": cc / t_one / 1e12, "cores": 1, "seconds_per_sample_apply": t_one},
            "host_cpus": os.cpu_count(), "cc_sample": cc}


def full_cc(cfg_name):
    """CC of the full workload counted in Python (oracle/cc_count.py), for the extrapolated full-apply time."""
    from gen import workloads as W
    from oracle.cc_count import cc_flops
    if cfg_name == "cfg1":
        return None
    return cc_flops(W.config_problem(cfg_name, seed=0, fill=False))[0]


def u1_equivalent(cfg_name):
    """The paper's rescaling to a U(1) calculation of the same accuracy (PAPER.md:231-241 Table I, :255): R_CC = CC of the
    operator written out in the (N, 2 S_z) basis with merged sectors / CC of the SU(2) plan, R_D = ratio of the bond
    dimensions.  The expansion is oracle-side (oracle/heff_u1.py, structure only); both CCs come from host-only plans."""
    from gen import workloads as W
    from oracle.heff_u1 import expand_problem
    from paper_2309_16724_b200 import Plan
    if cfg_name == "cfg1":
        return None
    prob = W.config_problem(cfg_name, seed=0, fill=False)
    u1, _ = expand_problem(prob, merged=True, with_data=False)
    cc_su2, cc_u1 = Plan(prob, host_only=True).info["cc_flops"], Plan(u1, host_only=True).info["cc_flops"]
    d_su2, d_u1 = sum(s.dim for s in prob.sec_l), sum(s.dim for s in u1.sec_l)
    return {"R_CC": cc_u1 / cc_su2, "R_D": d_u1 / d_su2, "D_SU2": d_su2, "D_U1": d_u1, "cc_flops_u1": cc_u1,
            "note": "U(1)-only mode of the same planner (SU2_SYMMETRY_U1) on the (N, 2Sz) expansion with merged sectors; "
                    "synthetic sector tables (windowed rule, S <= 2), so the ratios are those of this workload, not the paper's"}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only).  Loads nothing of the product."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cb = time_oracle(args.config, budget_s=30.0)
    cc_full = full_cc(args.config)
    extra = None if cc_full is None else cc_full / (cb["value"] * 1e12)
    line = {"metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * cb["seconds_per_sample_apply"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": args.config + " (oracle on a bounded sample)", "sample": cb["sample"],
                       "step": "one oracle H_eff*Psi on the sample (best of up to 3)",
                       "extrapolated_seconds_per_full_apply": extra},
            "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "single_thread", "host_cpus")},
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------ GPU arm
GANG_PACING = False      # --gang-pacing: plan flag SU2_PLAN_GANG_PACING (single-GPU operator)
TWO_PASS = {}            # --fused / --two-pass-...: plan flag SU2_PLAN_FUSED, options of the two-pass route (single-GPU operator)


def build_operator(cfg_name, device, shard=False):
    """Operator families resident in HBM, in the padded layout the large-tile kernel reads in place (ld_align = 4).
    cfg1-3: numpy counter-based generator, uploaded; cfg4 (92 GB): generated on the device (seeded torch generator,
    gen/device_ops.py), DESIGN.md "Input recipe".  shard=True: this rank's position slice of every family
    (paper_2309_16724_b200/sharding.py) under the current torch.distributed process group; the device generator
    reproduces the N = 1 operator's values at the positions a rank holds."""
    from gen import workloads as W
    from paper_2309_16724_b200.runtime import HeffOperator
    from paper_2309_16724_b200.sharding import ShardedHeffOperator, shard_problem
    big = cfg_name in ("cfg4", "cfg4p")
    prob = W.config_problem(cfg_name, seed=0, fill=not big)
    if not shard:
        fill = None
        if big:
            from gen.device_ops import device_fill
            fill = device_fill(prob)
        return prob, HeffOperator(prob, device=device, device_fill=fill, gang_pacing=GANG_PACING, **TWO_PASS)
    import torch.distributed as dist
    live = dist.is_available() and dist.is_initialized()
    rank, world = (dist.get_rank(), dist.get_world_size()) if live else (0, 1)
    fill = None
    if big:
        from gen.device_ops import device_fill
        fill = device_fill(shard_problem(prob, rank, world))
    return prob, ShardedHeffOperator(prob, device, device_fill=fill)


def reduce_vals(values, device, world, op="max"):
    """Max (or sum) over ranks of a list of numbers (the contract's max-over-ranks device time)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return [float(v) for v in t.cpu()]


def cublas_two_step(torch, A, X, B, Cm, alpha, args):
    """ms per call of T = A X; C += alpha T B^T as two strided-batched cuBLAS DGEMMs (torch.bmm / baddbmm_): the paper's scheme,
    timed as a yardstick beside su2_gemm_pair_batched (never on the product path)."""
    T = torch.empty(A.shape[0], A.shape[1], X.shape[2], dtype=torch.float64, device=A.device)
    Bt = B.transpose(1, 2)

    def call():
        torch.bmm(A, X, out=T)
        Cm.baddbmm_(T, Bt, alpha=alpha)
    for _ in range(2):
        call()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        call()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / args.steps


def heavy_shapes(cfg, top=12):
    """The `top` most flop-heavy task shapes (m, k, n, p) of a configuration (cfg5 sweeps them next to the
    square shapes): flops = positions x min(2mkn + 2mnp, 2knp + 2mkp) summed over the tasks of a host-only plan."""
    from gen.workloads import config_problem
    from paper_2309_16724_b200 import Plan
    prob = config_problem(cfg, fill=False)
    plan = Plan(prob, host_only=True)
    t = plan.export_tasks()
    dims = [(prob.sec_l[lab[0]].dim, prob.sec_r[lab[4]].dim) for lab in plan.labels]
    acc = {}
    for o, i, fl, fr in zip(t["out_sec"], t["in_sec"], t["fam_l"], t["fam_r"]):
        (m, p), (k, n) = dims[o], dims[i]
        npos = max(prob.fam_l[fl].npos if fl >= 0 else 1, prob.fam_r[fr].npos if fr >= 0 else 1)
        acc[(m, k, n, p)] = acc.get((m, k, n, p), 0.0) + npos * min(2.0 * m * k * n + 2.0 * m * n * p, 2.0 * k * n * p + 2.0 * m * k * p)
    total = sum(acc.values())
    return [(shape, f / total) for shape, f in sorted(acc.items(), key=lambda kv: -kv[1])[:top]]


def run_cfg5(args):
    """BASELINE.json configs[4]: strided-batched FP64 GEMM-pair microbenchmark, C_b += alpha A_b X_b B_b^T,
    square shapes 8..512, batch sized to ~1.5 GB of operands, through su2_gemm_pair_batched."""
    import torch
    from paper_2309_16724_b200 import gemm_pair_batched
    from paper_2309_16724_b200.binding import kernel_launch_count, probe_fp64_peak
    from paper_2309_16724_b200.build import build
    assert torch.cuda.is_available(), "bench.py needs a GPU (no CPU fallback)"
    build()
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    gen = torch.Generator(device="cuda").manual_seed(0)
    sweep = []
    l0 = kernel_launch_count()
    for b in (8, 16, 32, 64, 128, 256, 512):
        batch = int(max(1000, min(1000000, 1.5e9 / (4 * b * b * 8))))
        A, X, B, Cm = (torch.randn(batch, b, b, dtype=torch.float64, device="cuda", generator=gen) for _ in range(4))
        call = lambda: gemm_pair_batched(b, b, b, b, batch, 0.5, A.data_ptr(), X.data_ptr(), B.data_ptr(), Cm.data_ptr(), stream)
        for _ in range(max(3, args.warmup)):
            call()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            call()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        flops = 4.0 * b ** 3 * batch
        sweep.append({"m=k=n=p": b, "batch": batch, "ms": ms, "tflops": flops / ms / 1e9,
                      "operand_gbs": 8.0 * 5 * b * b * batch / ms / 1e6,
                      # yardstick, not part of the product: the paper's own scheme, two strided-batched vendor DGEMMs with
                      # T written to memory in between, through torch.bmm / baddbmm (cuBLAS)
                      "tflops_cublas_two_step": flops / cublas_two_step(torch, A, X, B, Cm, 0.5, args) / 1e9})
        del A, X, B, Cm
    # the most flop-heavy task shapes of configs[1..3]: FP64 route, the vendor yardstick, and for the
    # shapes of configs[2..3] the INT8 route
    from paper_2309_16724_b200.binding import gemm_pair_batched_i8
    heavy = []
    hws = torch.empty(2 << 30, dtype=torch.uint8, device="cuda")
    for cfg in ("cfg2", "cfg3", "cfg4"):
        for (m, k, n, p), share in heavy_shapes(cfg, args.heavy_shapes):
            batch = int(max(4, min(100000, 0.75e9 / (8.0 * (m * k + k * n + p * n + m * p)))))
            A = torch.randn(batch, m, k, dtype=torch.float64, device="cuda", generator=gen)
            X = torch.randn(batch, k, n, dtype=torch.float64, device="cuda", generator=gen)
            B = torch.randn(batch, p, n, dtype=torch.float64, device="cuda", generator=gen)
            Cm = torch.randn(batch, m, p, dtype=torch.float64, device="cuda", generator=gen)
            flops = (2.0 * m * k * n + 2.0 * m * n * p) * batch
            row = {"config": cfg, "m,k,n,p": [m, k, n, p], "flop_share_of_config": share, "batch": batch}
            routes = [("fp64", lambda: gemm_pair_batched(m, k, n, p, batch, 0.5, A.data_ptr(), X.data_ptr(), B.data_ptr(), Cm.data_ptr(), stream))]
            if cfg != "cfg2":
                routes.append(("i8", lambda: gemm_pair_batched_i8(m, k, n, p, batch, 0.5, A.data_ptr(), X.data_ptr(), B.data_ptr(),
                                                                  Cm.data_ptr(), stream, 7, hws.data_ptr(), hws.numel())))
            for name, call in routes:
                for _ in range(3):
                    call()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for _ in range(args.steps):
                    call()
                e1.record()
                torch.cuda.synchronize()
                row["tflops_" + name] = flops / (e0.elapsed_time(e1) / args.steps) / 1e9
            row["tflops_cublas_two_step"] = flops / cublas_two_step(torch, A, X, B, Cm, 0.5, args) / 1e9
            heavy.append(row)
            del A, X, B, Cm
    del hws
    # The same operation on the INT8 tensor path (include/su2_ozaki.h), next to the FP64 tensor route
    # on the same operands; 1024 and 2048 extend BASELINE.json's shape list to where the FP64 ceiling is passed.
    from paper_2309_16724_b200.binding import gemm_pair_batched_i8, ozaki_launch_count, ozaki_workspace_bytes
    sweep_i8 = []
    li0 = ozaki_launch_count()
    ws_bytes = 4 << 30
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
    for b in (128, 256, 512, 1024, 2048):
        batch = int(max(8, 1.5e9 / (4 * b * b * 8)))
        A, X, B, C8, C64 = (torch.randn(batch, b, b, dtype=torch.float64, device="cuda", generator=gen) for _ in range(5))
        C64.copy_(C8)
        row = {"m=k=n=p": b, "batch": batch, "nslices": 7,
               "items_per_chunk": min(batch, max(1, ws_bytes // ozaki_workspace_bytes(b, b, b, b, 1)))}
        for name, Cm, call in (("i8", C8, lambda: gemm_pair_batched_i8(b, b, b, b, batch, 0.5, A.data_ptr(), X.data_ptr(), B.data_ptr(),
                                                                      C8.data_ptr(), stream, 7, ws.data_ptr(), ws_bytes)),
                               ("fp64", C64, lambda: gemm_pair_batched(b, b, b, b, batch, 0.5, A.data_ptr(), X.data_ptr(), B.data_ptr(),
                                                                      C64.data_ptr(), stream))):
            call()                                     # the first call of each route on identical C: compared below
            if name == "fp64":
                row["max_diff_over_max_abs"] = float((C8 - C64).abs().max() / C64.abs().max())
            for _ in range(max(3, args.warmup)):
                call()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(args.steps):
                call()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / args.steps
            row["ms_" + name], row["tflops_" + name] = ms, 4.0 * b ** 3 * batch / ms / 1e9
            if name == "i8":                           # put C8 back to one call's worth for the comparison
                C8.copy_(C64)
                call()
        sweep_i8.append(row)
        del A, X, B, C8, C64
    del ws
    launches_i8 = ozaki_launch_count() - li0
    dmma = probe_fp64_peak(1, 4000, 4, stream)
    peaks, peak_src = measured_peaks()
    for r in sweep_i8:
        r["i8_over_fp64_tensor_peak"] = r["tflops_i8"] / dmma
    for r in sweep:   # algorithmic bytes per item: A, X, B read, C read + written (8 * 5 b^2)
        r["hbm_frac"] = r["operand_gbs"] / peaks["hbm_gbs"]
        r["tensor_frac"] = r["tflops"] / dmma
        r["bound"] = "hbm" if r["m=k=n=p"] / 10.0 < dmma * 1e3 / peaks["hbm_gbs"] else "tensor"
    best = max(sweep, key=lambda r: r["tflops"])
    best_hbm = max((r for r in sweep if r["bound"] == "hbm"), key=lambda r: r["operand_gbs"])
    print(json.dumps({"metric": METRIC, "value": best["tflops"], "unit": UNIT, "n_gpus": 1, "steps": args.steps,
                      "warmup": max(3, args.warmup), "ms_per_step": best["ms"], "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": "cfg5: strided-batched GEMM-pair microbenchmark (BASELINE.json configs[4]), square shapes; "
                                             "value = best shape", "l2": "operands 1.5 GB per shape exceed L2"},
                      "gpu_launches": kernel_launch_count() - l0 + launches_i8, "sweep": sweep, "heavy_task_shapes": heavy,
                      "int8_path": {"what": "the same GEMM pair by su2_gemm_pair_batched_i8: 7 INT8 slices of 7 bits, exact "
                                            "tcgen05 kind::i8 products, FP64 recombination (oracle/ozaki.py); tflops = 4 b^3 "
                                            "batch / time, the FP64-equivalent rate; NOT the line's value",
                                    "fp64_tensor_peak_measured": dmma, "gpu_launches": launches_i8, "sweep": sweep_i8},
                      "roofline": {"bound": "tensor", "achieved": best["tflops"], "peak": dmma, "unit": UNIT,
                                   "frac": best["tflops"] / dmma, "traffic": None},
                      "roofline_small_blocks": {"bound": "hbm", "kernel": "gemm_pair_small_kernel",
                                                "shape": best_hbm["m=k=n=p"], "achieved": best_hbm["operand_gbs"],
                                                "peak": peaks["hbm_gbs"], "peak_source": peak_src, "unit": "GB/s",
                                                "frac": best_hbm["hbm_frac"],
                                                "traffic": ncu_traffic("cfg5_b%d" % best_hbm["m=k=n=p"])}}))


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from gen.workloads import random_psi
    from paper_2309_16724_b200.binding import kernel_launch_count, probe_fp64_peak
    from paper_2309_16724_b200.build import build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    mode = args.parallelism or ("shard" if world > 1 else "single")
    if world > 1:
        if rank == 0:          # keep the communicator's own lines visible (transport, NVLS), on stderr
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT,ENV")
            os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        dist.init_process_group("nccl")
    assert torch.cuda.is_available(), "bench.py needs a GPU (no CPU fallback)"
    device = "cuda:%d" % local
    torch.cuda.set_device(device)
    if rank == 0:
        build()
    if world > 1:
        dist.barrier()
    stream = torch.cuda.current_stream().cuda_stream

    # FP64 tensor peak of this GPU, measured before the load (and again after it: the higher reading is the denominator;
    # right after a 1 kW run the short probe can catch a power-cap clock dip and read low, which would flatter frac)
    dmma_cold = probe_fp64_peak(1, 4000, 4, stream) if rank == 0 else 0.0
    t0 = time.perf_counter()
    prob, op = build_operator(args.config, device, shard=(mode == "shard"))
    setup_s = time.perf_counter() - t0
    local_op = op.local if mode == "shard" else op
    info = local_op.info
    cc_local = info["cc_flops"]
    # CC of the whole job: the shards add up to ONE operator; replicas are N operators
    cc_job = reduce_vals([cc_local], device, world, "sum")[0] if mode != "single" else cc_local
    psi0 = torch.from_numpy(random_psi(op.psi_len, seed=0)).to(device)
    solver = op.davidson(psi0, max_subspace=max(4, min(20, args.steps + args.warmup + 2)))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # --- warm-up
    hist = []
    for _ in range(args.warmup):
        hist.append(solver.step())
    # --- timed region: K Davidson steps, device time, max over ranks
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    l0 = kernel_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        hist.append(solver.step())
    ev1.record()
    barrier()
    launches = kernel_launch_count() - l0
    ms_total = ev0.elapsed_time(ev1)
    # --- the dominant kernel alone: the LOCAL su2_heff_apply (fused GEMM pair + reduction), CUDA events
    x, y = psi0.clone(), local_op.new_vector()
    ka0, ka1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    long_apply = ms_total / args.steps > 2000.0           # cfg4: one apply takes seconds
    napply = 1 if long_apply else max(1, min(args.steps, 5))
    if not long_apply:
        local_op.apply(x, y)
    torch.cuda.synchronize()
    ka0.record()
    for _ in range(napply):
        local_op.apply(x, y)
    ka1.record()
    torch.cuda.synchronize()
    apply_ms = ka0.elapsed_time(ka1) / napply
    # --- the same apply on the INT8 tensor path (su2_heff_apply_i8), on request: reported next to
    # the FP64 figure, never instead of it
    int8_path = None
    if args.int8_apply and mode == "single":
        from paper_2309_16724_b200.binding import ozaki_launch_count
        wsb = int(args.int8_workspace_gb * (1 << 30))
        y8 = local_op.apply_i8(x, workspace_bytes=wsb)          # warm-up (workspace allocation, first launches)
        torch.cuda.synchronize()
        diff = float((y8 - y).abs().max() / y.abs().max())
        n8 = 1 if long_apply else max(1, min(args.steps, 5))
        li0 = ozaki_launch_count()
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0.record()
        for _ in range(n8):
            local_op.apply_i8(x, y8, workspace_bytes=wsb)
        k1.record()
        torch.cuda.synchronize()
        ms8 = k0.elapsed_time(k1) / n8
        int8_path = {"what": "su2_heff_apply_i8: every task of the same plan as sliced exact INT8 products (7 slices), FP64 "
                             "recombination; FP64-equivalent rate = CC / time", "apply_ms": ms8,
                     "tflops": cc_local / (ms8 * 1e-3) / 1e12, "speedup_over_fp64_apply": apply_ms / ms8,
                     "max_diff_over_max_abs_vs_fp64_apply": diff, "gpu_launches_per_apply": (ozaki_launch_count() - li0) // n8,
                     "workspace_bytes": wsb}
    clocks = sampler.stop() if rank == 0 else None
    # --- end to end through the public API with HOST buffers (pinned): H2D psi, apply (+ all-reduce), D2H F, every step
    xh = psi0.cpu().pin_memory()
    fh = torch.empty_like(xh).pin_memory()
    if not long_apply:
        op.apply_host(xh, fh)
    barrier()
    t1 = time.perf_counter()
    ne2e = 1 if long_apply else max(1, min(args.steps, 5))
    for _ in range(ne2e):
        op.apply_host(xh, fh)
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t1) / ne2e

    ms_total, e2e_ms = reduce_vals([ms_total, e2e_ms], device, world, "max")
    if rank != 0:
        solver.close()
        if world > 1:
            dist.destroy_process_group()
        return

    ms_step = ms_total / args.steps
    peaks, peak_src = measured_peaks()
    dfma = probe_fp64_peak(0, 20000, 4, stream)
    dmma_hot = probe_fp64_peak(1, 4000, 4, stream)
    # third yardstick of SURVEY.md 8(d): the vendor DGEMM at 8192^3 (torch.matmul = cuBLAS; not part of the product)
    ga = torch.randn(8192, 8192, dtype=torch.float64, device=device)
    gb = torch.randn(8192, 8192, dtype=torch.float64, device=device)
    gc = torch.empty_like(ga)
    torch.matmul(ga, gb, out=gc)
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record()
    for _ in range(3):
        torch.matmul(ga, gb, out=gc)
    g1.record()
    torch.cuda.synchronize()
    cublas_dgemm = 3 * 2.0 * 8192.0 ** 3 / (g0.elapsed_time(g1) * 1e-3) / 1e12
    del ga, gb, gc
    dmma = max(dmma_cold, dmma_hot)
    peak = dmma
    peak_rule = peaks["bf16_tflops"] * FP64_OVER_BF16_NOMINAL
    achieved = cc_local / (apply_ms * 1e-3) / 1e12
    par_text = {"single": "single GPU",
                "shard": "positions sharded over %d rank(s), one FP64 all-reduce of F (%d bytes) per step" % (world, 8 * op.psi_len),
                "replicas": "%d independent replicas" % world}[mode]
    line = {
        "metric": METRIC, "value": cc_job / (ms_step * 1e-3) / 1e12, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "strong" if mode == "shard" else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: L=%d N=%d S=0 D_SU2=%d middle bond (BASELINE.json configs)" % (
                       args.config, prob.meta["L"], prob.meta["N"], prob.meta["D"]),
                   "step": "one su2_davidson_step = H_eff*Psi%s + Rayleigh-Ritz/residual/orthogonalisation" % (
                       " (local apply + all-reduce)" if mode == "shard" else ""),
                   "parallelism": par_text,
                   "l2": ("inputs exceed L2 (operators %.2f GB resident per rank, streamed every apply)" if local_op.operator_bytes_resident > 252e6
                          else "operators %.3f GB fit the 126 MB L2 and stay there between applies (not flushed): "
                               "small-block configuration, not the headline") % (local_op.operator_bytes_resident / 1e9),
                   "layout": "operator blocks with leading dimensions padded to a multiple of 4 (read in place by bulk-tensor copies)",
                   "gang_pacing": bool(GANG_PACING),
                   "two_pass": {"tasks": int(info["two_pass_tasks"]), "groups": int(info["two_pass_groups"]),
                                "scratch_bytes": int(info["two_pass_scratch_bytes"]), "options": TWO_PASS},
                   "small_plan": int(info["small_plan"]),
                   "psi_len": int(info["psi_len"]), "tasks": int(info["ntasks"]),
                   "task_positions": int(info["ntask_positions"]), "cc_flops_per_apply": cc_job,
                   "cc_flops_per_apply_this_rank": cc_local,
                   "executed_flops_per_apply_this_rank": info["executed_flops"], "work_items": int(info["nwork_items"]),
                   "segments": int(info["nsegments"]), "plan_seconds": info["plan_seconds"], "setup_seconds": setup_s,
                   "plan_device_bytes": int(info["plan_device_bytes"]), "padded_copy_bytes": int(info["padded_copy_bytes"])},
        "clocks": clocks,
        "e2e": {"value": cc_job / (e2e_ms * 1e-3) / 1e12, "unit": UNIT, "h2d_bytes_per_step": 8 * op.psi_len * world,
                "d2h_bytes_per_step": 8 * op.psi_len * world, "ms_per_step": e2e_ms,
                "call": "apply_host: pinned host Psi in, host F out (su2_heff_apply_host%s)" % (
                    "" if mode != "shard" else "-equivalent: H2D, su2_heff_apply, all-reduce, D2H")},
        "gpu_launches": int(launches),
        "roofline": {"bound": "tensor", "kernel": "%s = one su2_heff_apply on this rank" % (
                         "heff_small_kernel, one launch per size class (+reduce_kernel)" if info["small_plan"] else
                         "tp_gemm_kernel, %d launch groups of pass 1 + pass 2 (+tp_reduce_kernel)" % info["two_pass_groups"]
                         if info["two_pass_tasks"] else "heff_tma_kernel (+reduce_kernel)"),
                     "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                     "traffic": ncu_traffic(args.config),
                     "peak_source": "FP64 tensor (DMMA.8x8x4) loop measured in this run by su2_probe_fp64_peak (libsu2probe.so): "
                                    "max of the reading before the load (%.2f) and after it (%.2f)" % (dmma_cold, dmma_hot),
                     "peak_nominal": torch.cuda.get_device_properties(device).multi_processor_count * 128 *
                                     ((clocks or {}).get("sm_max_mhz") or 1965.0) * 1e-6,
                     "peak_bf16_ratio_rule": peak_rule, "frac_of_bf16_ratio_rule": achieved / peak_rule,
                     "peak_bf16_ratio_rule_source": "%s bf16_tflops x nominal FP64/BF16 ratio 45/2250" % peak_src,
                     "instruction_path": "FP64 tensor: mma.sync.m8n8k4.f64 = SASS DMMA.8x8x4; operands staged by cp.async.bulk.tensor (UTMALDG)",
                     "flops": "CC of the plan (useful flops, PAPER.md:229), not executed flops; achieved = CC / CUDA-event time of "
                              "the whole apply (all launches of the dominant kernel, back to back on one stream)",
                     "apply_ms": apply_ms, "launches_timed": napply, "peak_dfma_loop_measured": dfma,
                     "cublas_dgemm_8192_measured": cublas_dgemm,
                     "hbm_achieved_gbs": info["operator_bytes"] / (apply_ms * 1e-3) / 1e9, "hbm_peak_gbs": peaks["hbm_gbs"]},
        "davidson": {"theta": [h[0] for h in hist], "resnorm": [h[1] for h in hist]},
    }
    if int8_path is not None:
        int8_path["over_fp64_tensor_peak"] = int8_path["tflops"] / peak
        line["int8_path"] = int8_path
    if not args.no_cpu_baseline and world == 1:
        cb = time_oracle(args.config, budget_s=20.0)
        line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "single_thread", "host_cpus")}
        line["cpu_baseline"]["extrapolated_seconds_per_full_apply"] = cc_job / (cb["value"] * 1e12)
        u1 = u1_equivalent(args.config)
        if u1 is not None:       # reported NEXT TO the plain figure, never instead of it
            u1["u1_equivalent_tflops"] = line["value"] * u1["R_CC"]
            line["u1_equivalent"] = u1
    print(json.dumps(line))
    solver.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg4")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--heavy-shapes", type=int, default=12, help="cfg5: task shapes per configuration in the non-square sweep")
    ap.add_argument("--int8-apply", action="store_true",
                    help="also time H_eff*Psi on the INT8 tensor path (su2_heff_apply_i8) and report it as int8_path")
    ap.add_argument("--int8-workspace-gb", type=float, default=8.0)
    ap.add_argument("--gang-pacing", action="store_true",
                    help="plan with SU2_PLAN_GANG_PACING (row tiles of a sector paced for L2 reuse: less DRAM traffic, 2-5 %% slower)")
    ap.add_argument("--fused", action="store_true",
                    help="plan with SU2_PLAN_FUSED: every task on the fused large-tile kernel (default: the two-pass route, T through a plan-owned scratch)")
    ap.add_argument("--two-pass-min-dim", type=int, default=0)
    ap.add_argument("--two-pass-chunk-k", type=int, default=0)
    ap.add_argument("--two-pass-scratch-gb", type=float, default=0.0)
    ap.add_argument("--parallelism", default=None, choices=["shard", "replicas"],
                    help="N > 1: shard (default; one operator over N GPUs, strong scaling) or replicas (weak)")
    args = ap.parse_args()
    global GANG_PACING
    GANG_PACING = bool(args.gang_pacing)
    if args.fused:
        TWO_PASS.update(fused=True)
    elif args.two_pass_min_dim or args.two_pass_chunk_k or args.two_pass_scratch_gb:
        TWO_PASS.update(two_pass_min_dim=args.two_pass_min_dim, two_pass_chunk_k=args.two_pass_chunk_k,
                        two_pass_scratch_bytes=int(args.two_pass_scratch_gb * 2**30))
    if args.impl == "reference":
        run_reference(args)
        return
    if args.config == "cfg5":
        run_cfg5(args)
        return
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        # started plainly with --gpus N: become N ranks (one process per GPU) under torch.distributed.run
        import socket
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        sys.exit("bench.py: --gpus %d but WORLD_SIZE=%d: launch with --nproc-per-node equal to --gpus" % (args.gpus, world))
    run_gpu(args)


if __name__ == "__main__":
    main()
