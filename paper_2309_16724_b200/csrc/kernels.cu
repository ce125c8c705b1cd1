// Host side of su2_heff_apply and the small kernels around the fused GEMM pair (heff_dmma.cu):
//   reduce_kernel : second pass of the deterministic segmented reduction:
//                   fixed-order sum of the partial tiles of split sectors (no atomics).
//   diag_kernel   : diagonal of H_eff for the Davidson preconditioner.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstring>
#include <string>

#include <map>

#include "su2_internal.h"
#include "tile_config.h"

namespace su2 {

static thread_local std::string g_cuda_error;
static std::atomic<long long> g_launches{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
void set_cuda_error(const char* what, int code) {
  g_cuda_error = std::string(what) + ": " + cudaGetErrorString((cudaError_t)code);
}
void set_error_text(const char* what) { g_cuda_error = what; }
#define SU2_CUDA(call)                              \
  do {                                              \
    cudaError_t _e = (call);                        \
    if (_e != cudaSuccess) {                        \
      set_cuda_error(#call, (int)_e);               \
      return SU2_ERR_CUDA;                          \
    }                                               \
  } while (0)

// Second pass of the segmented reduction: fixed index order, one thread per element.
__global__ void __launch_bounds__(256)
reduce_kernel(const DevReduce* __restrict__ red, const double* __restrict__ partial, double* __restrict__ out) {
  const DevReduce r = red[blockIdx.y];
  if (r.nseg == 1) return;                    // written directly by the fused kernel
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < r.size; i += (int64_t)gridDim.x * blockDim.x) {
    double s = 0.0;
    for (int g = 0; g < r.nseg; ++g) s += partial[r.part_off + (int64_t)g * r.size + i];
    out[r.f_off + i] = s;
  }
}

// Plan-time position folding (the paper's pre-contraction): dst[r][c] = sum_pos alpha_pos src[pos][r][c],
// positions summed in index order (deterministic).  HBM-bound, runs once per plan.
__global__ void __launch_bounds__(256)
fold_kernel(const FoldJob* __restrict__ jobs, const double* __restrict__ alpha, double* __restrict__ fold) {
  const FoldJob j = jobs[blockIdx.y];
  const double* __restrict__ al = j.alpha_off >= 0 ? alpha + j.alpha_off : nullptr;
  const int64_t nelem = (int64_t)j.rows * j.cols, pstride = (int64_t)j.rows * j.ld_src;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < nelem; e += (int64_t)gridDim.x * blockDim.x) {
    const int r = (int)(e / j.cols), c = (int)(e % j.cols);
    const double* __restrict__ src = j.src + (int64_t)r * j.ld_src + c;
    double s = 0.0;
    for (int pos = 0; pos < j.npos; ++pos) s += (al ? al[pos] : 1.0) * src[(int64_t)pos * pstride];
    fold[j.dst_off + (int64_t)r * j.ld_dst + c] = s;
  }
}

// Plan-time padded copy of a block whose rows are not 16-byte aligned (see plan.cpp): leading dimension ld_src -> ld_dst,
// pad columns zeroed.  blockIdx.y = job, blockIdx.z strides positions.
__global__ void __launch_bounds__(256)
copy_kernel(const CopyJob* __restrict__ jobs, double* __restrict__ buf) {
  const CopyJob j = jobs[blockIdx.y];
  const int64_t nelem = (int64_t)j.rows * j.ld_dst;
  for (int pos = blockIdx.z; pos < j.npos; pos += gridDim.z) {
    const double* __restrict__ src = j.src + (int64_t)pos * j.rows * j.ld_src;
    double* __restrict__ dst = buf + j.dst_off + (int64_t)pos * nelem;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < nelem; e += (int64_t)gridDim.x * blockDim.x) {
      const int r = (int)(e / j.ld_dst), c = (int)(e % j.ld_dst);
      dst[e] = c < j.cols ? src[(int64_t)r * j.ld_src + c] : 0.0;
    }
  }
}

// Every apply of a large-tile plan: Psi -> the plan's padded private copy (rows on 32-byte boundaries) the E boxes
// are loaded from.  HBM-bound, 16 bytes per element of Psi: 0.05 ms at configs[3] against seconds of compute.
__global__ void __launch_bounds__(256)
psi_pad_kernel(const PsiPadJob* __restrict__ jobs, const double* __restrict__ psi, double* __restrict__ pad) {
  const PsiPadJob j = jobs[blockIdx.y];
  const int64_t nelem = (int64_t)j.rows * j.ld_dst;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < nelem; e += (int64_t)gridDim.x * blockDim.x) {
    const int r = (int)(e / j.ld_dst), c = (int)(e % j.ld_dst);
    pad[j.dst_off + e] = c < j.cols ? psi[j.src_off + (int64_t)r * j.cols + c] : 0.0;
  }
}

// diag(H_eff)[s][a,b] = sum_{tasks s<-s} coef sum_pos alpha_pos A_pos[a,a] D_pos[b,b]
__global__ void __launch_bounds__(256)
diag_kernel(const DevDiagTask* __restrict__ dt, const int32_t* __restrict__ begin, const PsiSector* __restrict__ psi_sec,
            double* __restrict__ diag) {
  const int s = blockIdx.y;
  const int m = psi_sec[s].m, p = psi_sec[s].p;
  const int64_t off = psi_sec[s].off;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < (int64_t)m * p; e += (int64_t)gridDim.x * blockDim.x) {
    const int a = (int)(e / p), b = (int)(e % p);
    double acc = 0.0;
    for (int i = begin[s]; i < begin[s + 1]; ++i) {
      const DevDiagTask t = dt[i];
      double v = 0.0;
      for (int pos = 0; pos < t.npos; ++pos) {
        const double al = t.alpha ? t.alpha[pos] : 1.0;
        v += al * t.A[(int64_t)pos * t.strideA + (int64_t)a * t.ldA + a] * t.D[(int64_t)pos * t.strideD + (int64_t)b * t.ldD + b];
      }
      acc += t.coef * v;
    }
    diag[off + e] = acc;
  }
}

// ---------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------
static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

namespace {
struct DeviceFree {   // frees on scope exit (error paths of upload_plan)
  void* p = nullptr;
  ~DeviceFree() { if (p) cudaFree(p); }
};
}  // namespace

su2_status upload_plan(su2_plan* plan, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  int dev = 0;
  SU2_CUDA(cudaGetDevice(&dev));
  SU2_CUDA(cudaDeviceGetAttribute(&plan->num_sms, cudaDevAttrMultiProcessorCount, dev));
  const bool large = plan->small_dm8 == 0;
  // ---- plan-owned operator buffers -------------------------------------------------------------
  auto big_alloc = [&](double** ptr, int64_t elems, const char* what) -> su2_status {
    if (elems <= 0) return SU2_OK;
    cudaError_t e = cudaMalloc((void**)ptr, (size_t)elems * sizeof(double));
    if (e != cudaSuccess) {   // fail loudly: there is no slower layout to fall back to
      *ptr = nullptr;
      char buf[200];
      std::snprintf(buf, sizeof(buf), "cudaMalloc of %.2f GB for %s", elems * 8.0 / 1e9, what);
      set_cuda_error(buf, (int)e);
      (void)cudaGetLastError();
      return SU2_ERR_CUDA;
    }
    plan->info.plan_device_bytes += elems * (int64_t)sizeof(double);
    return SU2_OK;
  };
  plan->info.plan_device_bytes = 0;
  su2_status st;
  if ((st = big_alloc(&plan->d_fold, plan->fold_elems, "the position-folded operators")) != SU2_OK) return st;
  if ((st = big_alloc(&plan->d_copy, plan->copy_elems,
                      "padded copies of operator families whose rows are not 16-byte aligned (pass blk_ld with even "
                      "leading dimensions to have them read in place)")) != SU2_OK) return st;
  if ((st = big_alloc(&plan->d_psi_pad, plan->psipad_elems, "the padded copy of Psi")) != SU2_OK) return st;
  if (!plan->tp_scratch_external &&
      (st = big_alloc(&plan->d_tp_scratch, plan->tp_scratch_elems,
                      "the scratch of the two-pass route (su2_plan_options.two_pass_scratch_bytes; or pass a caller-owned "
                      "buffer in two_pass_scratch_dev)")) != SU2_OK) return st;
  // a ragged k tail of T read as the right operand reaches into the rows of the next position: whatever is there is
  // multiplied by exact zeros, so it only has to be finite -- zero once (later contents are finite products)
  if (plan->d_tp_scratch) SU2_CUDA(cudaMemsetAsync(plan->d_tp_scratch, 0, (size_t)plan->tp_scratch_elems * sizeof(double), stream));

  // ---- resolve operand pointers; tensor maps of the large-tile kernel ------------------------------
  std::vector<unsigned char> h_maps;       // 128-byte records
  std::map<MapKey, int32_t> map_index;
  auto map_for = [&](const MapKey& key, int32_t* out) -> su2_status {
    auto it = map_index.find(key);
    if (it != map_index.end()) { *out = it->second; return SU2_OK; }
    const int32_t idx = (int32_t)map_index.size();
    h_maps.resize((size_t)(idx + 1) * 128);
    su2_status s2 = encode_tensor_map(h_maps.data() + (size_t)idx * 128, key);
    if (s2 != SU2_OK) return s2;
    map_index[key] = idx;
    *out = idx;
    return SU2_OK;
  };
  const size_t b_tasks = align256(plan->h_tasks.size() * sizeof(DevTask));
  const size_t b_units = align256(plan->h_units.size() * sizeof(DevUnit));
  const size_t b_work = align256(plan->h_work.size() * sizeof(DevWork));
  const size_t b_red = align256(plan->h_reduce.size() * sizeof(DevReduce));
  const size_t b_diag = align256(plan->h_diag.size() * sizeof(DevDiagTask));
  const size_t b_dbeg = align256(plan->h_diag_begin.size() * sizeof(int32_t));
  const size_t b_psi = align256(plan->psi.size() * sizeof(PsiSector));
  const size_t b_pad = align256(plan->h_psipad.size() * sizeof(PsiPadJob));
  const size_t b_alpha = align256(plan->h_alpha.size() * sizeof(double));
  const size_t b_ident = align256(plan->h_ident.size() * sizeof(double));
  // the identity blocks must exist before their tensor maps are encoded: allocate the blob first (maps are
  // appended to it in a second allocation-free step: their count is bounded by 3 per task)
  // (+ the two-pass route: at most 4 per slice)
  const size_t b_maps = align256(large ? (3 * plan->h_tasks.size() + 4 * plan->h_tp_slices.size() + 1) * 128 : 0);
  const size_t b_tps = align256(plan->h_tp_slices.size() * sizeof(TpSlice));
  const size_t b_tpr = align256(plan->h_tp_reduce.size() * sizeof(TpReduce));
  const size_t b_gang = align256((size_t)plan->n_gang_slots * sizeof(int32_t));
  const size_t total = b_tasks + b_units + b_work + b_red + b_diag + b_dbeg + b_psi + b_pad + b_alpha + b_ident + b_maps + b_gang + b_tps + b_tpr + 256;
  SU2_CUDA(cudaMalloc(&plan->d_blob, total));
  plan->info.plan_device_bytes += (int64_t)total;
  char* base = (char*)plan->d_blob;
  size_t off = 0;
  auto carve = [&](size_t bytes) { char* q = base + off; off += bytes; return q; };
  plan->d_maps = carve(b_maps);            // first: 256-byte aligned records
  plan->d_tasks = (DevTask*)carve(b_tasks);
  plan->d_units = (DevUnit*)carve(b_units);
  plan->d_work = (DevWork*)carve(b_work);
  plan->d_reduce = (DevReduce*)carve(b_red);
  plan->d_diag = (DevDiagTask*)carve(b_diag);
  plan->d_diag_begin = (int32_t*)carve(b_dbeg);
  char* d_psi = carve(b_psi);
  plan->d_psipad = (PsiPadJob*)carve(b_pad);
  plan->d_alpha = (double*)carve(b_alpha);
  plan->d_identity = (double*)carve(b_ident);
  plan->d_counter = (int32_t*)carve(256);
  plan->d_gang = b_gang ? (int32_t*)carve(b_gang) : nullptr;
  plan->d_tp_slices = (TpSlice*)carve(b_tps);
  plan->d_tp_reduce = (TpReduce*)carve(b_tpr);

  auto resolve = [&](const OperandRef& r) -> const double* {
    switch (r.kind) {
      case 0: { const double* b0 = plan->fam_ptr[r.side][r.fam]; return b0 ? b0 + r.off : nullptr; }
      case 1: return plan->d_copy ? plan->d_copy + r.off : nullptr;
      case 2: return plan->d_fold ? plan->d_fold + r.off : nullptr;
      default: return plan->d_identity + r.off;
    }
  };
  for (size_t i = 0; i < plan->h_tasks.size(); ++i) {
    DevTask& t = plan->h_tasks[i];
    const OperandRef &ra = plan->h_opA[i], &rd = plan->h_opD[i];
    t.A = resolve(ra);
    t.D = resolve(rd);
    if (!t.A || !t.D) return SU2_ERR_INVALID_ARGUMENT;   // family without device data
    if (plan->h_alpha_off[i] >= 0) t.alpha = plan->d_alpha + plan->h_alpha_off[i];
    if (!large || plan->tasks[i].two_pass) continue;
    const int wr = plan->tasks[i].wr;
    const int tm = 32 * wr;
    MapKey ka{t.A, ra.rows, ra.cols, ra.ld, ra.npos, (int64_t)ra.rows * ra.ld,
              (t.flags & TASK_TRANS_A) ? tm + 4 : KS1, (t.flags & TASK_TRANS_A) ? KS1 : tm};
    MapKey kd{t.D, rd.rows, rd.cols, rd.ld, rd.npos, (int64_t)rd.rows * rd.ld,
              (t.flags & TASK_TRANS_D) ? DBOX_LD : KS2, (t.flags & TASK_TRANS_D) ? KS2 : DBOX_C};
    const PsiPadJob& pj = plan->h_psipad[plan->tasks[i].in_sec];
    MapKey ke{plan->d_psi_pad + pj.dst_off, pj.rows, pj.cols, pj.ld_dst, 1, (int64_t)pj.rows * pj.ld_dst, EBOX_LD, KS1};
    if ((st = map_for(ka, &t.mapA)) != SU2_OK || (st = map_for(kd, &t.mapD)) != SU2_OK || (st = map_for(ke, &t.mapE)) != SU2_OK) return st;
    t.e_item = 0;
  }
  // two-pass route: tensor maps with the boxes of tp_gemm_kernel (heff_two_pass.cu)
  for (TpSlice& sl : plan->h_tp_slices) {
    const DevTask& t = plan->h_tasks[sl.task];
    const OperandRef &ra = plan->h_opA[sl.task], &rd = plan->h_opD[sl.task];
    const bool ta = t.flags & TASK_TRANS_A, td = t.flags & TASK_TRANS_D;
    // Aop is always the left operand: as stored (rows x k boxes) or read transposed (k x rows boxes)
    MapKey ka{t.A, ra.rows, ra.cols, ra.ld, ra.npos, (int64_t)ra.rows * ra.ld, ta ? TP_LLD : TP_KS, ta ? TP_KS : TP_TM};
    // Dop^T is always the right operand: D stored p x n has the inner index contiguous, stored n x p the columns
    MapKey kd{t.D, rd.rows, rd.cols, rd.ld, rd.npos, (int64_t)rd.rows * rd.ld, td ? TP_RLD : TP_KS, td ? TP_KS : TP_TN};
    // E (k x n): right operand of A E (columns contiguous), left operand of E D^T (as stored)
    const PsiPadJob& pj = plan->h_psipad[plan->tasks[sl.task].in_sec];
    MapKey ke{plan->d_psi_pad + pj.dst_off, pj.rows, pj.cols, pj.ld_dst, 1, (int64_t)pj.rows * pj.ld_dst, sl.order ? TP_KS : TP_RLD,
              sl.order ? TP_TM : TP_KS};
    // T: the scratch as one matrix of rows of ldt doubles, colsT of them valid; left operand of T D^T, right operand of A T
    const int colsT = sl.order ? t.p : t.n;
    const int64_t rows_all = plan->tp_scratch_elems / sl.ldt;
    if (rows_all > 0x7fffffff) { set_error_text("two-pass scratch too large for 32-bit row coordinates"); return SU2_ERR_INVALID_ARGUMENT; }
    MapKey kt{plan->d_tp_scratch, (int32_t)rows_all, colsT, sl.ldt, 1, rows_all * sl.ldt, sl.order ? TP_RLD : TP_KS, sl.order ? TP_KS : TP_TM};
    if ((st = map_for(ka, &sl.mapA)) != SU2_OK || (st = map_for(kd, &sl.mapD)) != SU2_OK || (st = map_for(ke, &sl.mapE)) != SU2_OK ||
        (st = map_for(kt, &sl.mapT)) != SU2_OK)
      return st;
  }
  plan->nmaps = (int32_t)map_index.size();
  for (auto& d : plan->h_diag) {
    const DevTask& t = plan->h_tasks[d.pad];
    d.A = t.A; d.D = t.D; d.alpha = t.alpha;
  }
  auto up = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
    if (bytes == 0) return cudaSuccess;
    return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, stream);
  };
  SU2_CUDA(up(plan->d_maps, h_maps.data(), h_maps.size()));
  SU2_CUDA(up(plan->d_tasks, plan->h_tasks.data(), plan->h_tasks.size() * sizeof(DevTask)));
  SU2_CUDA(up(plan->d_units, plan->h_units.data(), plan->h_units.size() * sizeof(DevUnit)));
  SU2_CUDA(up(plan->d_work, plan->h_work.data(), plan->h_work.size() * sizeof(DevWork)));
  SU2_CUDA(up(plan->d_reduce, plan->h_reduce.data(), plan->h_reduce.size() * sizeof(DevReduce)));
  SU2_CUDA(up(plan->d_diag, plan->h_diag.data(), plan->h_diag.size() * sizeof(DevDiagTask)));
  SU2_CUDA(up(plan->d_diag_begin, plan->h_diag_begin.data(), plan->h_diag_begin.size() * sizeof(int32_t)));
  SU2_CUDA(up(d_psi, plan->psi.data(), plan->psi.size() * sizeof(PsiSector)));
  SU2_CUDA(up(plan->d_psipad, plan->h_psipad.data(), plan->h_psipad.size() * sizeof(PsiPadJob)));
  SU2_CUDA(up(plan->d_alpha, plan->h_alpha.data(), plan->h_alpha.size() * sizeof(double)));
  SU2_CUDA(up(plan->d_identity, plan->h_ident.data(), plan->h_ident.size() * sizeof(double)));
  SU2_CUDA(up(plan->d_tp_slices, plan->h_tp_slices.data(), plan->h_tp_slices.size() * sizeof(TpSlice)));
  SU2_CUDA(up(plan->d_tp_reduce, plan->h_tp_reduce.data(), plan->h_tp_reduce.size() * sizeof(TpReduce)));
  DeviceFree d_fjobs, d_cjobs;
  if (plan->fold_elems > 0) {
    for (const FoldJob& j : plan->h_fold)
      if (!j.src) return SU2_ERR_INVALID_ARGUMENT;   // family without device data
    SU2_CUDA(cudaMalloc(&d_fjobs.p, plan->h_fold.size() * sizeof(FoldJob)));
    SU2_CUDA(cudaMemcpyAsync(d_fjobs.p, plan->h_fold.data(), plan->h_fold.size() * sizeof(FoldJob), cudaMemcpyHostToDevice, stream));
    SU2_CUDA(cudaMemsetAsync(plan->d_fold, 0, (size_t)plan->fold_elems * sizeof(double), stream));   // pad columns
    dim3 grid(64, (unsigned)plan->h_fold.size());
    fold_kernel<<<grid, 256, 0, stream>>>((const FoldJob*)d_fjobs.p, plan->d_alpha, plan->d_fold);
    SU2_CUDA(cudaGetLastError());
    count_launch();
  }
  if (plan->copy_elems > 0) {
    for (const CopyJob& j : plan->h_copy)
      if (!j.src) return SU2_ERR_INVALID_ARGUMENT;
    SU2_CUDA(cudaMalloc(&d_cjobs.p, plan->h_copy.size() * sizeof(CopyJob)));
    SU2_CUDA(cudaMemcpyAsync(d_cjobs.p, plan->h_copy.data(), plan->h_copy.size() * sizeof(CopyJob), cudaMemcpyHostToDevice, stream));
    dim3 grid(64, (unsigned)plan->h_copy.size(), 16);
    copy_kernel<<<grid, 256, 0, stream>>>((const CopyJob*)d_cjobs.p, plan->d_copy);
    SU2_CUDA(cudaGetLastError());
    count_launch();
  }
  SU2_CUDA(cudaStreamSynchronize(stream));
  plan->d_psi_sec = d_psi;
  plan->info.padded_copy_bytes = plan->copy_elems * (int64_t)sizeof(double);
  return SU2_OK;
}

void free_plan_device(su2_plan* plan) {
  if (!plan) return;
  if (plan->tp_scratch_external) plan->d_tp_scratch = nullptr;   // caller-owned
  for (void** q : {(void**)&plan->d_blob, (void**)&plan->d_fold, (void**)&plan->d_copy, (void**)&plan->d_psi_pad, (void**)&plan->d_tp_scratch})
    if (*q) { cudaFree(*q); *q = nullptr; }
}

su2_status launch_apply(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  SU2_CUDA(cudaMemsetAsync(plan->d_counter, 0, 8 * sizeof(int32_t), stream));   // [0]: work queue; small plans: one per size class
  su2_status st;
  if (plan->small_dm8 > 0) {
    st = launch_heff_small(plan, psi, out, partial, stream_v);
  } else {
    if (!plan->h_psipad.empty()) {
      dim3 grid(16, (unsigned)plan->h_psipad.size());
      psi_pad_kernel<<<grid, 256, 0, stream>>>(plan->d_psipad, psi, plan->d_psi_pad);
      SU2_CUDA(cudaGetLastError());
      count_launch();
    }
    if (plan->d_gang)   // pacing slots: -1 = member not started
      SU2_CUDA(cudaMemsetAsync(plan->d_gang, 0xff, (size_t)plan->n_gang_slots * sizeof(int32_t), stream));
    st = plan->h_work.empty() ? SU2_OK : launch_heff_tma(plan, out, partial, stream_v);   // nothing left on the fused kernel
  }
  if (st != SU2_OK) return st;
  const int nsec = (int)plan->h_reduce.size();
  if (nsec > 0) {
    dim3 grid(32, nsec);
    reduce_kernel<<<grid, 256, 0, stream>>>(plan->d_reduce, partial, out);
    SU2_CUDA(cudaGetLastError());
    count_launch();
  }
  // tasks on the two-pass route add their share to `out` (partial slabs behind the fused kernel's partial tiles)
  if (!plan->h_tp_groups.empty()) {
    double* tp_partial = (double*)((char*)partial + align256((size_t)plan->partial_elems * 8 + 256));
    if ((st = launch_heff_two_pass(plan, out, tp_partial, stream_v)) != SU2_OK) return st;
  }
  return SU2_OK;
}

su2_status launch_diag(const su2_plan* plan, double* diag, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  const int nsec = (int)plan->psi.size();
  if (nsec == 0) return SU2_OK;
  dim3 grid(64, nsec);
  diag_kernel<<<grid, 256, 0, stream>>>(plan->d_diag, plan->d_diag_begin, (const PsiSector*)plan->d_psi_sec, diag);
  SU2_CUDA(cudaGetLastError());
  count_launch();
  return SU2_OK;
}

}  // namespace su2

using namespace su2;

extern "C" const char* su2_last_cuda_error(void) { return g_cuda_error.c_str(); }
extern "C" int64_t su2_kernel_launch_count(void) { return (int64_t)g_launches.load(std::memory_order_relaxed); }

extern "C" su2_status su2_heff_apply(const su2_plan* plan, const double* psi_dev, double* out_dev, void* workspace_dev,
                                     void* cuda_stream) {
  if (!plan || !psi_dev || !out_dev || psi_dev == out_dev) return SU2_ERR_INVALID_ARGUMENT;
  if (plan->host_only) return SU2_ERR_NO_DEVICE_PLAN;
  if ((plan->partial_elems > 0 || plan->tp_partial_elems > 0) && !workspace_dev) return SU2_ERR_WORKSPACE;
  return launch_apply(plan, psi_dev, out_dev, (double*)workspace_dev, cuda_stream);
}

extern "C" su2_status su2_heff_apply_host(const su2_plan* plan, const double* psi_host, double* out_host,
                                          void* workspace_dev, void* cuda_stream) {
  if (!plan || !psi_host || !out_host) return SU2_ERR_INVALID_ARGUMENT;
  if (plan->host_only) return SU2_ERR_NO_DEVICE_PLAN;
  if (!workspace_dev) return SU2_ERR_WORKSPACE;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace_dev;
  const size_t wsb = (size_t)plan->info.workspace_bytes;
  double* d_psi = (double*)(ws + ((wsb + 255) & ~(size_t)255));
  double* d_out = d_psi + plan->psi_len;
  SU2_CUDA(cudaMemcpyAsync(d_psi, psi_host, plan->psi_len * sizeof(double), cudaMemcpyHostToDevice, stream));
  su2_status st = launch_apply(plan, d_psi, d_out, (double*)workspace_dev, cuda_stream);
  if (st != SU2_OK) return st;
  SU2_CUDA(cudaMemcpyAsync(out_host, d_out, plan->psi_len * sizeof(double), cudaMemcpyDeviceToHost, stream));
  SU2_CUDA(cudaStreamSynchronize(stream));
  return SU2_OK;
}

extern "C" su2_status su2_heff_diag(const su2_plan* plan, double* diag_dev, void* cuda_stream) {
  if (!plan || !diag_dev) return SU2_ERR_INVALID_ARGUMENT;
  if (plan->host_only) return SU2_ERR_NO_DEVICE_PLAN;
  return launch_diag(plan, diag_dev, cuda_stream);
}
