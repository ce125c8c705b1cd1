"""PyTorch-side plumbing around the C ABI: device memory for operator families, Psi and the
workspace, and the CUDA stream.  No arithmetic of the hot path happens here: apply(), diag()
and the Davidson steps run inside libsu2heff.so; a missing extension or GPU raises."""
import numpy as np
import torch

from .binding import Davidson, Plan, Su2Error, family_layout


def _require_cuda():
    if not torch.cuda.is_available():
        raise Su2Error("no CUDA device: the product path has no CPU fallback")


class HeffOperator:
    """H_eff of one superblock problem, resident on one GPU.

    problem: gen.problem.Problem-like plain data.  Family data is taken from
    problem.fam_*[i].data (list of numpy blocks [npos, m, k]) or, when `device_fill` is given,
    generated directly on the device by device_fill(side, index, tensor) (143 GB-class
    workloads cannot be staged through host memory)."""

    def __init__(self, problem, device="cuda:0", device_fill=None, force_split=False, large_tiles=False, ld_align=4, gang_pacing=False,
                 fused=False, two_pass=False, **two_pass_opts):
        """fused: plan flag SU2_PLAN_FUSED (every task on the fused kernel; default: large-tile plans run un-fused through a
        plan-owned scratch, SU2_PLAN_TWO_PASS); two_pass_opts: two_pass_min_dim, two_pass_chunk_k, two_pass_scratch_bytes
        (su2_plan_options).
        ld_align: leading dimensions of the operator blocks in device memory are rounded up to this multiple
        (binding.family_layout).  4 (default) puts every row on a 32-byte boundary, so that the large-tile kernel
        reads the operators in place with bulk-tensor copies; 1 is the dense layout, of which the plan makes a
        padded copy when it needs one."""
        _require_cuda()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.problem = problem
        self.ld_align = ld_align
        self.family_tensors = {}
        self.family_layouts = {}
        ptrs = {}
        for side, fams, secs in (("l", problem.fam_l, problem.sec_l), ("r", problem.fam_r, problem.sec_r)):
            for i, f in enumerate(fams):
                offs, lds, n = family_layout(f, secs, ld_align)
                self.family_layouts[(side, i)] = (offs, lds)
                if device_fill is not None:
                    t = torch.empty(max(n, 1), dtype=torch.float64, device=self.device)
                    device_fill(side, i, t, offs, lds)
                else:
                    host = np.zeros(max(n, 1))
                    for b, (off, ld) in zip(f.data, zip(offs, lds)):
                        npos, m, k = b.shape
                        host[off:off + npos * m * ld].reshape(npos, m, ld)[:, :, :k] = b
                    t = torch.from_numpy(host).to(self.device)
                self.family_tensors[(side, i)] = t
                ptrs[(side, i)] = t.data_ptr()
        self.stream = torch.cuda.current_stream(self.device)
        # The scratch of the two-pass route is a torch tensor (PyTorch owns every large allocation; the plan gets its address
        # through su2_plan_options.two_pass_scratch_dev).  Its size is what the plan itself would take: asked of a host-only
        # plan with the same flags and options first.  two_pass_scratch="library": the plan allocates it itself.
        self.two_pass_scratch = None
        if two_pass_opts.pop("two_pass_scratch", "torch") == "torch" and not fused and not gang_pacing:
            probe = Plan(problem, family_ptrs=None, host_only=True, force_split=force_split, large_tiles=large_tiles, ld_align=ld_align,
                         two_pass=two_pass, **two_pass_opts)
            nbytes = int(probe.info["two_pass_scratch_bytes"])
            del probe
            if nbytes > 0:
                self.two_pass_scratch = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
                two_pass_opts = dict(two_pass_opts, two_pass_scratch_bytes=nbytes, two_pass_scratch_ptr=self.two_pass_scratch.data_ptr())
        self.plan = Plan(problem, family_ptrs=ptrs, stream=self.stream.cuda_stream, force_split=force_split,
                         large_tiles=large_tiles, ld_align=ld_align, gang_pacing=gang_pacing, fused=fused, two_pass=two_pass, **two_pass_opts)
        self.psi_len = self.plan.psi_len
        # workspace: partial tiles + staging for the host entry point
        self.workspace = torch.empty(self.plan.workspace_bytes + 16 * self.psi_len, dtype=torch.uint8,
                                     device=self.device)
        self.operator_bytes_resident = sum(t.numel() * 8 for t in self.family_tensors.values())

    @property
    def info(self):
        return self.plan.info

    def new_vector(self):
        return torch.empty(self.psi_len, dtype=torch.float64, device=self.device)

    def apply(self, psi, out=None):
        """out = H_eff psi (device tensors, float64, contiguous)."""
        assert psi.dtype == torch.float64 and psi.is_cuda and psi.is_contiguous() and psi.numel() == self.psi_len
        if out is None:
            out = self.new_vector()
        self.plan.heff_apply(psi.data_ptr(), out.data_ptr(), self.workspace.data_ptr(),
                             torch.cuda.current_stream(self.device).cuda_stream)
        return out

    def apply_noalloc(self, psi, out):
        """out = H_eff psi through su2_heff_apply_noalloc: no workspace, nothing allocated (caller passes both tensors)."""
        assert psi.dtype == torch.float64 and psi.is_cuda and psi.is_contiguous() and psi.numel() == self.psi_len
        assert out.dtype == torch.float64 and out.is_cuda and out.is_contiguous() and out.numel() == self.psi_len
        self.plan.heff_apply_noalloc(psi.data_ptr(), out.data_ptr(), torch.cuda.current_stream(self.device).cuda_stream)
        return out

    def apply_i8(self, psi, out=None, nslices=0, workspace_bytes=4 << 30):
        """out = H_eff psi with every task on the INT8 tensor path (su2_heff_apply_i8, include/su2_ozaki.h): the same
        plan and operands, executed as sliced exact integer products; the workspace is allocated on first use."""
        from .binding import heff_apply_i8
        assert psi.dtype == torch.float64 and psi.is_cuda and psi.is_contiguous() and psi.numel() == self.psi_len
        if out is None:
            out = torch.empty(self.psi_len, dtype=torch.float64, device=self.device)
        if getattr(self, "_i8_views", None) is None:
            self._i8_views = self.plan.export_task_views()
        if getattr(self, "_i8_ws", None) is None or self._i8_ws.numel() < workspace_bytes:
            self._i8_ws = torch.empty(workspace_bytes, dtype=torch.uint8, device=self.device)
        heff_apply_i8(self._i8_views, psi.data_ptr(), out.data_ptr(), self.psi_len, self._i8_ws.data_ptr(), workspace_bytes,
                      torch.cuda.current_stream(self.device).cuda_stream, nslices)
        return out

    def apply_host(self, psi_host, out_host):
        """End-to-end entry: pinned host tensors in and out (copies inside the C call)."""
        assert psi_host.dtype == torch.float64 and not psi_host.is_cuda and psi_host.numel() == self.psi_len
        self.plan.heff_apply_host(psi_host.data_ptr(), out_host.data_ptr(), self.workspace.data_ptr(),
                                  torch.cuda.current_stream(self.device).cuda_stream)
        return out_host

    def diag(self):
        d = self.new_vector()
        self.plan.heff_diag(d.data_ptr(), torch.cuda.current_stream(self.device).cuda_stream)
        return d

    def davidson(self, x0, max_subspace=20):
        return DavidsonSolver(self, x0, max_subspace)


class DavidsonSolver:
    def __init__(self, op, x0, max_subspace=20):
        self.op = op
        nbytes = Davidson.workspace_bytes(op.plan, max_subspace)
        self.ws = torch.empty(nbytes, dtype=torch.uint8, device=op.device)
        self.stream = torch.cuda.current_stream(op.device).cuda_stream
        self.dav = Davidson(op.plan, max_subspace, x0.data_ptr(), self.ws.data_ptr(), self.stream)
        self.history = []

    def step(self):
        theta, res = self.dav.step(self.op.workspace.data_ptr(), self.stream)
        self.history.append((theta, res))
        return theta, res

    def ritz_vector(self):
        x = self.op.new_vector()
        self.dav.ritz_vector(x.data_ptr(), self.stream)
        return x

    def close(self):
        self.dav.close()


def precontract_family(fam, secs, weights, device="cuda:0", ld_align=4):
    """Complementary family from a normal one on the device (su2_precontract): `fam` is a gen.problem.OpFamily-like object
    with numpy blocks [npos, m, k], `weights` a (npos_out x npos) array.  Returns the list of output blocks
    [npos_out, m, k] as numpy arrays (marshalling only: the contraction runs in the library)."""
    from .binding import family_layout, precontract
    _require_cuda()
    dev = torch.device(device)
    w = np.ascontiguousarray(weights, dtype=np.float64)
    npos_out, npos_in = w.shape
    assert npos_in == fam.npos
    offs_in, lds, n_in = family_layout(fam, secs, ld_align)
    host = np.zeros(max(n_in, 1))
    elems, offs_out, cur = [], [], 0
    for b, (blk, off, ld) in enumerate(zip(fam.data, offs_in, lds)):
        _, m, k = blk.shape
        host[off:off + npos_in * m * ld].reshape(npos_in, m, ld)[:, :, :k] = blk
        elems.append(m * ld)
        offs_out.append(cur)
        cur += -(-npos_out * m * ld // 16) * 16
    d_in = torch.from_numpy(host).to(dev)
    d_w = torch.from_numpy(w).to(dev)
    d_out = torch.zeros(max(cur, 1), dtype=torch.float64, device=dev)
    precontract(elems, offs_in, offs_out, npos_in, npos_out, d_w.data_ptr(), d_in.data_ptr(), d_out.data_ptr(),
                torch.cuda.current_stream(dev).cuda_stream)
    out_host = d_out.cpu().numpy()
    out = []
    for blk, off, ld in zip(fam.data, offs_out, lds):
        _, m, k = blk.shape
        out.append(out_host[off:off + npos_out * m * ld].reshape(npos_out, m, ld)[:, :, :k].copy())
    return out


def renormalize_family(sec_old, sec_new, channels, rotation, fam_old, site, twoK_new, new_blocks, weight=1.0,
                       device="cuda:0", ld_align=4):
    """Blocking step on the device (su2_renormalize): the operator [O_l x O_B]^{k'} of the enlarged block in its new basis.

    sec_old / sec_new: lists of (N, twoS, dim); channels[q'] = [(block sector, site multiplet, first row)] (the coupled
    rows of new sector q'); rotation[q'] = numpy (coupled rows x D') matrix; fam_old: OpFamily-like with numpy blocks
    [npos, m, k] over sec_old, or None (identity); site: SiteOp-like (r, dN, twoK) or None; new_blocks: list of
    (q'_out, q'_in) to compute.  Returns the list of new blocks [npos, D'_out, D'_in] as numpy arrays (marshalling only)."""
    from types import SimpleNamespace
    from .binding import family_layout, renormalize
    _require_cuda()
    dev = torch.device(device)
    stream = torch.cuda.current_stream(dev).cuda_stream
    # rotation matrices, padded leading dimensions, one buffer
    u_off, u_ld, cur = [], [], 0
    for q, (_, _, d) in enumerate(sec_new):
        ld = -(-d // ld_align) * ld_align
        u_off.append(cur)
        u_ld.append(ld)
        cur += -(-rotation[q].shape[0] * ld // 16) * 16
    u_host = np.zeros(max(cur, 1))
    for q, (_, _, d) in enumerate(sec_new):
        rows = rotation[q].shape[0]
        u_host[u_off[q]:u_off[q] + rows * u_ld[q]].reshape(rows, u_ld[q])[:, :d] = rotation[q]
    d_u = torch.from_numpy(u_host).to(dev)
    chan = [(q, il, sg, r0) for q, lst in enumerate(channels) for (il, sg, r0) in lst]
    old = None
    npos, dN, kl = 1, 0, 0
    if fam_old is not None:
        secs = [SimpleNamespace(N=s[0], twoS=s[1], dim=s[2]) for s in sec_old]
        offs, lds, n = family_layout(fam_old, secs, ld_align)
        host = np.zeros(max(n, 1))
        for blk, off, ld in zip(fam_old.data, offs, lds):
            p_, m, k = blk.shape
            host[off:off + p_ * m * ld].reshape(p_, m, ld)[:, :, :k] = blk
        d_old = torch.from_numpy(host).to(dev)
        npos, dN, kl = fam_old.npos, fam_old.dN, fam_old.twoK
        old = dict(dN=dN, twoK=kl, npos=npos, q_out=fam_old.q_out, q_in=fam_old.q_in, offs=offs, lds=lds, ptr=d_old.data_ptr())
    dN_new = dN + (site.dN if site is not None else 0)
    secs_new = [SimpleNamespace(N=s[0], twoS=s[1], dim=s[2]) for s in sec_new]
    new_fam = SimpleNamespace(npos=npos, q_out=[b[0] for b in new_blocks], q_in=[b[1] for b in new_blocks])
    offs_n, lds_n, n_new = family_layout(new_fam, secs_new, ld_align)
    d_new = torch.full((max(n_new, 1),), float("nan"), dtype=torch.float64, device=dev)   # must be overwritten / zeroed
    new = dict(dN=dN_new, twoK=twoK_new, npos=npos, q_out=new_fam.q_out, q_in=new_fam.q_in, offs=offs_n, lds=lds_n,
               ptr=d_new.data_ptr())
    renormalize(sec_old, sec_new, chan, u_off, u_ld, d_u.data_ptr(), old,
                None if site is None else (site.r, site.dN, site.twoK), twoK_new, weight, False, new, stream)
    host_new = d_new.cpu().numpy()
    out = []
    for (qo, qi), off, ld in zip(new_blocks, offs_n, lds_n):
        m, k = sec_new[qo][2], sec_new[qi][2]
        out.append(host_new[off:off + npos * m * ld].reshape(npos, m, ld)[:, :, :k].copy())
    return out
