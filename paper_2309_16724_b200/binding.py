"""Thin Python binding of the C ABI in include/su2_heff.h (argument marshalling only: every
step of the hot path runs inside libsu2heff.so).  PyTorch is used by the callers for device
memory and streams; this module itself only needs ctypes + numpy."""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsu2heff.so")


class Su2Error(RuntimeError):
    pass


class su2_sector(C.Structure):
    _fields_ = [("N", C.c_int32), ("twoS", C.c_int32), ("dim", C.c_int32)]


class su2_opfamily(C.Structure):
    _fields_ = [("dN", C.c_int32), ("twoK", C.c_int32), ("npos", C.c_int32), ("nblk", C.c_int32),
                ("q_out", C.POINTER(C.c_int32)), ("q_in", C.POINTER(C.c_int32)),
                ("blk_off", C.POINTER(C.c_int64)), ("blk_ld", C.POINTER(C.c_int32)), ("data", C.c_void_p)]


class su2_siteop(C.Structure):
    _fields_ = [("r", (C.c_double * 3) * 3), ("dN", C.c_int32), ("twoK", C.c_int32)]


class su2_siteop_u1(C.Structure):
    _fields_ = [("r", (C.c_double * 4) * 4), ("dN", C.c_int32), ("dM", C.c_int32)]


class su2_blocking(C.Structure):
    _fields_ = [("nsec_old", C.c_int32), ("sec_old", C.POINTER(su2_sector)), ("nsec_new", C.c_int32),
                ("sec_new", C.POINTER(su2_sector)), ("nchan", C.c_int32), ("chan_new", C.POINTER(C.c_int32)),
                ("chan_old", C.POINTER(C.c_int32)), ("chan_site", C.POINTER(C.c_int32)), ("chan_row0", C.POINTER(C.c_int32)),
                ("u_off", C.POINTER(C.c_int64)), ("u_ld", C.POINTER(C.c_int32)), ("u", C.c_void_p)]


class su2_term(C.Structure):
    _fields_ = [("fam_l", C.c_int32), ("fam_r", C.c_int32), ("op_B", C.c_int32), ("op_C", C.c_int32),
                ("twoK_L", C.c_int32), ("twoK_R", C.c_int32), ("adj_l", C.c_int32), ("adj_r", C.c_int32),
                ("npos", C.c_int32), ("alpha", C.POINTER(C.c_double))]


class su2_problem(C.Structure):
    _fields_ = [("n_tot", C.c_int32), ("twoS_tot", C.c_int32), ("nsec_l", C.c_int32), ("nsec_r", C.c_int32),
                ("sec_l", C.POINTER(su2_sector)), ("sec_r", C.POINTER(su2_sector)),
                ("nfam_l", C.c_int32), ("nfam_r", C.c_int32),
                ("fam_l", C.POINTER(su2_opfamily)), ("fam_r", C.POINTER(su2_opfamily)),
                ("nsite", C.c_int32), ("site", C.POINTER(su2_siteop)),
                ("nterm", C.c_int32), ("term", C.POINTER(su2_term)),
                ("symmetry", C.c_int32), ("site_u1", C.POINTER(su2_siteop_u1))]


class su2_task_view(C.Structure):
    _fields_ = [("A", C.c_void_p), ("D", C.c_void_p), ("alpha", C.c_void_p), ("coef", C.c_double),
                ("strideA", C.c_int64), ("strideD", C.c_int64), ("e_off", C.c_int64), ("f_off", C.c_int64),
                ("ldA", C.c_int32), ("ldD", C.c_int32), ("transA", C.c_int32), ("transD", C.c_int32),
                ("m", C.c_int32), ("k", C.c_int32), ("n", C.c_int32), ("p", C.c_int32), ("npos", C.c_int32), ("pad", C.c_int32)]


class su2_plan_info_t(C.Structure):
    _fields_ = [("psi_len", C.c_int64), ("ntasks", C.c_int64), ("ntask_positions", C.c_int64),
                ("cc_flops", C.c_double), ("executed_flops", C.c_double), ("operator_bytes", C.c_double),
                ("workspace_bytes", C.c_int64), ("npsi_sec", C.c_int32), ("nsegments", C.c_int32),
                ("nwork_items", C.c_int64), ("plan_seconds", C.c_double), ("plan_device_bytes", C.c_int64),
                ("small_plan", C.c_int32), ("gang_slots", C.c_int32), ("padded_copy_bytes", C.c_int64),
                ("two_pass_tasks", C.c_int64), ("two_pass_scratch_bytes", C.c_int64), ("two_pass_groups", C.c_int32), ("pad", C.c_int32)]


class su2_plan_options(C.Structure):
    _fields_ = [("two_pass_min_dim", C.c_int32), ("two_pass_chunk_k", C.c_int32), ("two_pass_scratch_bytes", C.c_int64),
                ("two_pass_ipc_k", C.c_int32), ("pad", C.c_int32), ("two_pass_scratch_dev", C.c_void_p)]


EXPORTS = ["su2_wigner_6j", "su2_wigner_9j", "su2_status_string", "su2_last_cuda_error", "su2_kernel_launch_count", "su2_plan_create", "su2_plan_create_opts", "su2_plan_destroy", "su2_plan_info",
           "su2_plan_psi_layout", "su2_plan_export_tasks", "su2_heff_apply", "su2_heff_apply_host", "su2_heff_diag",
           "su2_davidson_workspace_bytes", "su2_davidson_create", "su2_davidson_create_sharded", "su2_davidson_step", "su2_davidson_set_preconditioner", "su2_davidson_ritz_vector",
           "su2_davidson_destroy", "su2_gemm_pair_batched", "su2_gemm_pair_batched_route", "su2_precontract", "su2_renormalize", "su2_heff_apply_noalloc",
           "su2_noalloc_scratch_bytes", "su2_plan_export_task_views"]

REDUCE_FN = C.CFUNCTYPE(C.c_int32, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p)   # su2_reduce_fn

SU2_PLAN_HOST_ONLY = 1
_lib = None


def load():
    """Load libsu2heff.so.  Fails loudly if the extension has not been built: there is no
    fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise Su2Error("CUDA extension %s is missing: run __graft_entry__.build() "
                       "(python -m paper_2309_16724_b200.build)" % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    for name in EXPORTS:
        getattr(lib, name).restype = C.c_int32
    lib.su2_wigner_6j.restype = C.c_double
    lib.su2_wigner_6j.argtypes = [C.c_int32] * 6
    lib.su2_wigner_9j.restype = C.c_double
    lib.su2_wigner_9j.argtypes = [C.c_int32] * 9
    lib.su2_status_string.restype = C.c_char_p
    lib.su2_status_string.argtypes = [C.c_int32]
    lib.su2_last_cuda_error.restype = C.c_char_p
    lib.su2_kernel_launch_count.restype = C.c_int64
    lib.su2_plan_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(su2_problem), C.c_int32, C.c_void_p]
    lib.su2_plan_create_opts.argtypes = [C.POINTER(C.c_void_p), C.POINTER(su2_problem), C.c_int32, C.POINTER(su2_plan_options), C.c_void_p]
    lib.su2_plan_destroy.argtypes = [C.c_void_p]
    lib.su2_plan_info.argtypes = [C.c_void_p, C.POINTER(su2_plan_info_t)]
    lib.su2_plan_psi_layout.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.su2_plan_export_tasks.argtypes = [C.c_void_p] + [C.c_void_p] * 10
    lib.su2_plan_export_task_views.restype = C.c_int64
    lib.su2_plan_export_task_views.argtypes = [C.c_void_p, C.POINTER(su2_task_view), C.c_int64]
    lib.su2_heff_apply.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.su2_heff_apply_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.su2_noalloc_scratch_bytes.restype = C.c_int64
    lib.su2_noalloc_scratch_bytes.argtypes = []
    lib.su2_heff_apply_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.su2_heff_diag.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.su2_davidson_workspace_bytes.restype = C.c_int64
    lib.su2_davidson_workspace_bytes.argtypes = [C.c_void_p, C.c_int32]
    lib.su2_davidson_create.argtypes = [C.POINTER(C.c_void_p), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.su2_davidson_create_sharded.argtypes = [C.POINTER(C.c_void_p), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p,
                                                C.c_void_p, REDUCE_FN, C.c_void_p]
    lib.su2_davidson_step.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.su2_davidson_set_preconditioner.argtypes = [C.c_void_p, C.c_int32]
    lib.su2_davidson_ritz_vector.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.su2_davidson_destroy.argtypes = [C.c_void_p]
    lib.su2_gemm_pair_batched.argtypes = [C.c_int32] * 4 + [C.c_int64, C.c_double] + [C.c_void_p] * 5
    lib.su2_gemm_pair_batched_route.argtypes = [C.c_int32] * 4 + [C.c_int64, C.c_double] + [C.c_void_p] * 5 + [C.c_int32] * 3
    lib.su2_precontract.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p,
                                    C.c_void_p, C.c_void_p, C.c_void_p]
    lib.su2_renormalize.argtypes = [C.POINTER(su2_blocking), C.POINTER(su2_opfamily), C.POINTER(su2_siteop), C.c_int32,
                                    C.c_double, C.c_int32, C.POINTER(su2_opfamily), C.c_void_p]
    _lib = lib
    return lib


def check(st):
    if st != 0:
        lib = load()
        msg = lib.su2_status_string(st).decode()
        if st in (-5, -8):
            msg += " (" + lib.su2_last_cuda_error().decode() + ")"
        raise Su2Error("su2 status %d: %s" % (st, msg))


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def family_layout(fam, secs, ld_align=1):
    """Layout of a family's device buffer: block b = [npos][dim(q_out)][ld_b] row-major with ld_b = dim(q_in) rounded up
    to a multiple of ld_align, blocks one after the other, every block starting on a multiple of 16 elements when
    ld_align > 1.  Returns (offsets, lds, total_elements).  ld_align = 1 is the dense layout; ld_align = 4 puts every
    row on a 32-byte boundary, which lets the large-tile kernel read the family in place (su2_heff.h)."""
    offs, lds, cur = [], [], 0
    for qo, qi in zip(fam.q_out, fam.q_in):
        offs.append(cur)
        if 0 <= qo < len(secs) and 0 <= qi < len(secs):      # bad indices are rejected by su2_plan_create
            ld = -(-secs[qi].dim // ld_align) * ld_align
            lds.append(ld)
            cur += fam.npos * secs[qo].dim * ld
            if ld_align > 1:
                cur = -(-cur // 16) * 16
        else:
            lds.append(1)
    return offs, lds, cur


def family_block_offsets(fam, secs):
    return family_layout(fam, secs)[0]


def family_elems(fam, secs):
    return family_layout(fam, secs)[2]


class Plan:
    """su2_plan wrapper.  `problem` is a gen.problem.Problem-like object (plain data);
    `family_ptrs` maps ("l"|"r", family index) -> DEVICE base pointer (int) of the family's
    blocks laid out as family_layout(fam, secs, ld_align) says; None for a host-only plan (planner tests
    without a GPU)."""

    def __init__(self, problem, family_ptrs=None, stream=0, host_only=False, force_split=False, large_tiles=False, gang_pacing=False,
                 ld_align=1, fused=False, two_pass=False, two_pass_min_dim=0, two_pass_chunk_k=0, two_pass_scratch_bytes=0, two_pass_ipc_k=0, two_pass_scratch_ptr=None):
        lib = load()
        self._keep = []
        self.problem = problem

        def sectors(secs):
            arr = (su2_sector * len(secs))(*[su2_sector(s.N, s.twoS, s.dim) for s in secs])
            self._keep.append(arr)
            return arr

        def families(fams, secs, side):
            arr = (su2_opfamily * max(len(fams), 1))()
            for i, f in enumerate(fams):
                qo, qi = _i32(f.q_out), _i32(f.q_in)
                offs, lds, _ = family_layout(f, secs, ld_align)
                off, ld = np.asarray(offs, dtype=np.int64), _i32(lds)
                self._keep += [qo, qi, off, ld]
                ptr = None if family_ptrs is None else family_ptrs[(side, i)]
                ldp = C.POINTER(C.c_int32)() if ld_align == 1 else ld.ctypes.data_as(C.POINTER(C.c_int32))
                arr[i] = su2_opfamily(f.dN, f.twoK, f.npos, len(f.q_out),
                                      qo.ctypes.data_as(C.POINTER(C.c_int32)), qi.ctypes.data_as(C.POINTER(C.c_int32)),
                                      off.ctypes.data_as(C.POINTER(C.c_int64)), ldp, ptr)
            self._keep.append(arr)
            return arr

        sl, sr = sectors(problem.sec_l), sectors(problem.sec_r)
        fl = families(problem.fam_l, problem.sec_l, "l")
        fr = families(problem.fam_r, problem.sec_r, "r")
        u1 = getattr(problem, "symmetry", "su2") == "u1"
        site = ((su2_siteop_u1 if u1 else su2_siteop) * len(problem.site))()
        for i, o in enumerate(problem.site):
            for a in range(4 if u1 else 3):
                for b in range(4 if u1 else 3):
                    site[i].r[a][b] = float(o.r[a][b])
            if u1:
                site[i].dN, site[i].dM = o.dN, o.twoK
            else:
                site[i].dN, site[i].twoK = o.dN, o.twoK
        terms = (su2_term * max(len(problem.term), 1))()
        for i, t in enumerate(problem.term):
            npos = problem.npos_of(t)
            if t.alpha is None:
                ap = C.POINTER(C.c_double)()
            else:
                a = np.ascontiguousarray(t.alpha, dtype=np.float64)
                assert a.shape == (npos,), (t.name, a.shape, npos)
                self._keep.append(a)
                ap = a.ctypes.data_as(C.POINTER(C.c_double))
            terms[i] = su2_term(t.fam_l, t.fam_r, t.op_B, t.op_C, t.twoK_L, t.twoK_R, t.adj_l, t.adj_r, npos, ap)
        self._keep += [site, terms]
        prob = su2_problem(problem.n_tot, problem.twoS_tot, len(problem.sec_l), len(problem.sec_r), sl, sr,
                           len(problem.fam_l), len(problem.fam_r), fl, fr, len(problem.site),
                           None if u1 else site, len(problem.term), terms, 1 if u1 else 0, site if u1 else None)
        self.handle = C.c_void_p()
        flags = ((SU2_PLAN_HOST_ONLY if host_only else 0) | (2 if force_split else 0) | (4 if large_tiles else 0) | (8 if gang_pacing else 0) |
                 (16 if two_pass else 0) | (32 if fused else 0))
        opts = su2_plan_options(int(two_pass_min_dim), int(two_pass_chunk_k), int(two_pass_scratch_bytes), int(two_pass_ipc_k), 0, two_pass_scratch_ptr)
        check(lib.su2_plan_create_opts(C.byref(self.handle), C.byref(prob), flags, C.byref(opts), C.c_void_p(stream)))
        info = su2_plan_info_t()
        check(lib.su2_plan_info(self.handle, C.byref(info)))
        self.info = {k: getattr(info, k) for k, _ in su2_plan_info_t._fields_}
        n = self.info["npsi_sec"]
        labels = np.zeros((n, 6), dtype=np.int32)
        offsets = np.zeros(n + 1, dtype=np.int64)
        check(lib.su2_plan_psi_layout(self.handle, labels.ctypes.data, offsets.ctypes.data))
        self.labels = [tuple(int(x) for x in row) for row in labels]
        self.offsets = offsets
        self.psi_len = int(self.info["psi_len"])
        self.workspace_bytes = int(self.info["workspace_bytes"])

    def export_tasks(self):
        n = int(self.info["ntasks"])
        names = ["out_sec", "in_sec", "fam_l", "blk_l", "adj_l", "fam_r", "blk_r", "adj_r", "term"]
        arrs = {k: np.zeros(n, dtype=np.int32) for k in names}
        coef = np.zeros(n, dtype=np.float64)
        check(load().su2_plan_export_tasks(self.handle, *[arrs[k].ctypes.data for k in names], coef.ctypes.data))
        arrs["coef"] = coef
        return arrs

    def export_task_views(self):
        """The uploaded task table with resolved device operands (su2_plan_export_task_views): a ctypes array of
        su2_task_view, valid as long as the plan lives."""
        n = int(load().su2_plan_export_task_views(self.handle, None, 0))
        if n < 0:
            raise Su2Error("su2_plan_export_task_views: host-only plan")
        views = (su2_task_view * n)()
        load().su2_plan_export_task_views(self.handle, views, n)
        return views

    # --- device entry points (pointers are plain ints) ---
    def heff_apply(self, psi_ptr, out_ptr, workspace_ptr, stream=0):
        check(load().su2_heff_apply(self.handle, psi_ptr, out_ptr, workspace_ptr, stream))

    def heff_apply_noalloc(self, psi_ptr, out_ptr, stream=0):
        """su2_heff_apply_noalloc: scratch in the library's static device array (<= 64 MiB), nothing allocated."""
        check(load().su2_heff_apply_noalloc(self.handle, psi_ptr, out_ptr, stream))

    def heff_apply_host(self, psi_host_ptr, out_host_ptr, workspace_ptr, stream=0):
        check(load().su2_heff_apply_host(self.handle, psi_host_ptr, out_host_ptr, workspace_ptr, stream))

    def heff_diag(self, diag_ptr, stream=0):
        check(load().su2_heff_diag(self.handle, diag_ptr, stream))

    def close(self):
        if getattr(self, "handle", None):
            load().su2_plan_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Davidson:
    def __init__(self, plan, max_subspace, x0_ptr, ws_ptr, stream=0, reduce=None):
        """reduce(vec_ptr, n, stream) -> status: sum over ranks of a device vector (position-sharded plans).
        An exception raised inside the hook is stored, reported to the library as a negative status (the C call
        stops there instead of continuing on an un-reduced vector) and re-raised from the Python call."""
        self.plan = plan
        self.handle = C.c_void_p()
        self._hook_error = None
        if reduce is None:
            check(load().su2_davidson_create(C.byref(self.handle), plan.handle, max_subspace, x0_ptr, ws_ptr, stream))
        else:
            def thunk(vec, n, st, user):
                try:
                    return int(reduce(vec, n, st) or 0)
                except BaseException as exc:          # never let an exception escape into ctypes
                    self._hook_error = exc
                    return -5
            self._reduce = REDUCE_FN(thunk)           # keep the thunk alive
            st = load().su2_davidson_create_sharded(C.byref(self.handle), plan.handle, max_subspace, x0_ptr, ws_ptr,
                                                    stream, self._reduce, None)
            self._raise_hook_error()
            check(st)

    def _raise_hook_error(self):
        if self._hook_error is not None:
            exc, self._hook_error = self._hook_error, None
            raise exc

    @staticmethod
    def workspace_bytes(plan, max_subspace):
        return int(load().su2_davidson_workspace_bytes(plan.handle, max_subspace))

    def step(self, workspace_ptr, stream=0):
        th, rn = C.c_double(), C.c_double()
        st = load().su2_davidson_step(self.plan.handle, self.handle, workspace_ptr, stream, C.byref(th), C.byref(rn))
        self._raise_hook_error()
        check(st)
        return th.value, rn.value

    def set_preconditioner(self, mode):
        check(load().su2_davidson_set_preconditioner(self.handle, int(mode)))

    def ritz_vector(self, x_ptr, stream=0):
        check(load().su2_davidson_ritz_vector(self.handle, x_ptr, stream))

    def close(self):
        if getattr(self, "handle", None):
            load().su2_davidson_destroy(self.handle)
            self.handle = C.c_void_p()


def gemm_pair_batched(m, k, n, p, batch, alpha, a_ptr, x_ptr, b_ptr, c_ptr, stream=0, route=0, wpi=0, nbuf=0):
    """route 0: automatic; 1: small-block kernel; 2: fused large-tile kernel; 3: FP64-FMA tile routine; 4: un-fused two-pass kernel."""
    if route == 0 and wpi == 0 and nbuf == 0:
        check(load().su2_gemm_pair_batched(m, k, n, p, batch, alpha, a_ptr, x_ptr, b_ptr, c_ptr, stream))
    else:
        check(load().su2_gemm_pair_batched_route(m, k, n, p, batch, alpha, a_ptr, x_ptr, b_ptr, c_ptr, stream, route, wpi, nbuf))


_probe = None


def probe_fp64_peak(kind, iters=20000, ctas_per_sm=4, stream=0):
    """Measured register-resident FP64 TFLOP/s: kind 0 = DFMA loop, 1 = DMMA.8x8x4 loop.  Lives in its own library
    (libsu2probe.so, include/su2_probe.h): a measurement aid of bench.py, not part of the product ABI."""
    global _probe
    if _probe is None:
        path = os.path.join(HERE, "libsu2probe.so")
        if not os.path.exists(path):
            raise Su2Error("%s is missing: run python -m paper_2309_16724_b200.build" % path)
        _probe = C.CDLL(path)
        _probe.su2_probe_fp64_peak.restype = C.c_int32
        _probe.su2_probe_fp64_peak.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_double), C.c_void_p]
    v = C.c_double()
    st = _probe.su2_probe_fp64_peak(kind, iters, ctas_per_sm, C.byref(v), stream)
    if st != 0:
        raise Su2Error("su2_probe_fp64_peak failed with status %d" % st)
    return v.value


def precontract(block_elems, in_off, out_off, npos_in, npos_out, w_ptr, in_ptr, out_ptr, stream=0):
    """out[b][pos'] = sum_pos W[pos'][pos] in[b][pos] for every block b (su2_precontract): host offset arrays, device data."""
    be = np.ascontiguousarray(block_elems, dtype=np.int64)
    io = np.ascontiguousarray(in_off, dtype=np.int64)
    oo = np.ascontiguousarray(out_off, dtype=np.int64)
    check(load().su2_precontract(len(be), be.ctypes.data, io.ctypes.data, oo.ctypes.data, npos_in, npos_out, w_ptr, in_ptr,
                                 out_ptr, stream))


def _family_struct(dN, twoK, npos, q_out, q_in, offs, lds, ptr, keep):
    qo, qi, off, ld = _i32(q_out), _i32(q_in), np.ascontiguousarray(offs, dtype=np.int64), _i32(lds)
    keep += [qo, qi, off, ld]
    return su2_opfamily(dN, twoK, npos, len(qo), qo.ctypes.data_as(C.POINTER(C.c_int32)), qi.ctypes.data_as(C.POINTER(C.c_int32)),
                        off.ctypes.data_as(C.POINTER(C.c_int64)), ld.ctypes.data_as(C.POINTER(C.c_int32)), ptr)


def renormalize(sec_old, sec_new, channels, u_off, u_ld, u_ptr, old, site, twoK_new, weight, accumulate, new, stream=0):
    """su2_renormalize.  sec_old / sec_new: lists of (N, twoS, dim); channels: list of (new sector, block sector, site
    multiplet, first row); old / new: None or dict(dN, twoK, npos, q_out, q_in, offs, lds, ptr) describing a family in
    DEVICE memory; site: None or (r 3x3, dN, twoK)."""
    keep = []
    so = (su2_sector * len(sec_old))(*[su2_sector(*s) for s in sec_old])
    sn = (su2_sector * len(sec_new))(*[su2_sector(*s) for s in sec_new])
    ch = [_i32([c[i] for c in channels]) for i in range(4)]
    uo, ul = np.ascontiguousarray(u_off, dtype=np.int64), _i32(u_ld)
    blk = su2_blocking(len(sec_old), so, len(sec_new), sn, len(channels), *[a.ctypes.data_as(C.POINTER(C.c_int32)) for a in ch],
                       uo.ctypes.data_as(C.POINTER(C.c_int64)), ul.ctypes.data_as(C.POINTER(C.c_int32)), u_ptr)
    f_old = None if old is None else _family_struct(old["dN"], old["twoK"], old["npos"], old["q_out"], old["q_in"], old["offs"],
                                                    old["lds"], old["ptr"], keep)
    f_new = _family_struct(new["dN"], new["twoK"], new["npos"], new["q_out"], new["q_in"], new["offs"], new["lds"], new["ptr"], keep)
    s_op = None
    if site is not None:
        s_op = su2_siteop()
        for a in range(3):
            for b in range(3):
                s_op.r[a][b] = float(site[0][a][b])
        s_op.dN, s_op.twoK = site[1], site[2]
    check(load().su2_renormalize(C.byref(blk), None if f_old is None else C.byref(f_old), None if s_op is None else C.byref(s_op),
                                 twoK_new, weight, 1 if accumulate else 0, C.byref(f_new), stream))


def wigner_6j(*two_j):
    return float(load().su2_wigner_6j(*[int(x) for x in two_j]))


def wigner_9j(*two_j):
    return float(load().su2_wigner_9j(*[int(x) for x in two_j]))


def noalloc_scratch_bytes():
    return int(load().su2_noalloc_scratch_bytes())


def kernel_launch_count():
    return int(load().su2_kernel_launch_count())


# ---- include/su2_ozaki.h: the GEMM pair on the INT8 tensor path (libsu2ozaki.so) ----------------------------
OZAKI_LIB_PATH = os.path.join(HERE, "libsu2ozaki.so")
_ozaki = None


def load_ozaki():
    global _ozaki
    if _ozaki is None:
        if not os.path.exists(OZAKI_LIB_PATH):
            raise Su2Error("%s is missing: run python -m paper_2309_16724_b200.build" % OZAKI_LIB_PATH)
        lib = C.CDLL(OZAKI_LIB_PATH)
        dp = C.c_void_p
        lib.su2_gemm_pair_batched_i8.restype = C.c_int32
        lib.su2_gemm_pair_batched_i8.argtypes = [C.c_int32] * 4 + [C.c_int64, C.c_double, dp, dp, dp, dp, C.c_int32, dp, C.c_size_t, dp]
        lib.su2_matmul_batched_i8.restype = C.c_int32
        lib.su2_matmul_batched_i8.argtypes = [C.c_int32] * 3 + [C.c_int64, dp, dp, dp, C.c_int32, dp, C.c_size_t, dp]
        lib.su2_heff_apply_i8.restype = C.c_int32
        lib.su2_heff_apply_i8.argtypes = [C.POINTER(su2_task_view), C.c_int64, dp, dp, C.c_int64, C.c_int32, dp, C.c_size_t, dp]
        lib.su2_ozaki_workspace_bytes.restype = C.c_size_t
        lib.su2_ozaki_workspace_bytes.argtypes = [C.c_int32] * 4 + [C.c_int64, C.c_int32]
        lib.su2_ozaki_launch_count.restype = C.c_int64
        lib.su2_ozaki_launch_count.argtypes = []
        lib.su2_ozaki_last_error.restype = C.c_char_p
        lib.su2_ozaki_last_error.argtypes = []
        _ozaki = lib
    return _ozaki


def _check_ozaki(st):
    if st != 0:
        raise Su2Error("su2_ozaki status %d: %s" % (st, load_ozaki().su2_ozaki_last_error().decode()))


def gemm_pair_batched_i8(m, k, n, p, batch, alpha, a_ptr, x_ptr, b_ptr, c_ptr, stream=0, nslices=0, workspace_ptr=None,
                         workspace_bytes=0):
    """C_b += alpha A_b X_b B_b^T on the INT8 tensor path (su2_gemm_pair_batched_i8): device pointers, dense strides."""
    _check_ozaki(load_ozaki().su2_gemm_pair_batched_i8(m, k, n, p, batch, alpha, a_ptr, x_ptr, b_ptr, c_ptr, nslices, workspace_ptr,
                                                       workspace_bytes, stream))


def matmul_batched_i8(m, k, n, batch, a_ptr, x_ptr, c_ptr, stream=0, nslices=0, workspace_ptr=None, workspace_bytes=0):
    """C_b = A_b X_b on the INT8 tensor path (su2_matmul_batched_i8)."""
    _check_ozaki(load_ozaki().su2_matmul_batched_i8(m, k, n, batch, a_ptr, x_ptr, c_ptr, nslices, workspace_ptr, workspace_bytes, stream))


def ozaki_workspace_bytes(m, k, n, p, items, nslices=0):
    return int(load_ozaki().su2_ozaki_workspace_bytes(m, k, n, p, items, nslices))


def ozaki_launch_count():
    return int(load_ozaki().su2_ozaki_launch_count())


def heff_apply_i8(task_views, psi_ptr, out_ptr, psi_len, workspace_ptr, workspace_bytes, stream=0, nslices=0):
    """out = H_eff psi with every task on the INT8 tensor path (su2_heff_apply_i8); task_views: Plan.export_task_views()."""
    _check_ozaki(load_ozaki().su2_heff_apply_i8(task_views, len(task_views), psi_ptr, out_ptr, psi_len, nslices, workspace_ptr,
                                                workspace_bytes, stream))
