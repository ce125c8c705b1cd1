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

    def __init__(self, problem, device="cuda:0", device_fill=None, force_split=False, large_tiles=False, ld_align=4):
        """ld_align: leading dimensions of the operator blocks in device memory are rounded up to this multiple
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
        self.plan = Plan(problem, family_ptrs=ptrs, stream=self.stream.cuda_stream, force_split=force_split,
                         large_tiles=large_tiles, ld_align=ld_align)
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
