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

#include "su2_internal.h"

namespace su2 {

static thread_local std::string g_cuda_error;
static std::atomic<long long> g_launches{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
void set_cuda_error(const char* what, int code) {
  g_cuda_error = std::string(what) + ": " + cudaGetErrorString((cudaError_t)code);
}
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

// Plan-time position folding (the paper's pre-contraction): dst[e] = sum_pos alpha_pos src[pos][e],
// positions summed in index order (deterministic).  HBM-bound, runs once per plan.
__global__ void __launch_bounds__(256)
fold_kernel(const FoldJob* __restrict__ jobs, const double* __restrict__ alpha, double* __restrict__ fold) {
  const FoldJob j = jobs[blockIdx.y];
  const double* __restrict__ al = j.alpha_off >= 0 ? alpha + j.alpha_off : nullptr;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < j.nelem; e += (int64_t)gridDim.x * blockDim.x) {
    double s = 0.0;
    for (int pos = 0; pos < j.npos; ++pos) s += (al ? al[pos] : 1.0) * j.src[(int64_t)pos * j.nelem + e];
    fold[j.dst_off + e] = s;
  }
}

// Plan-time transposed copy of a right-block operator block, 32x32 tiles through shared memory:
// dst[pos][j][c] = src[pos][c][j].  blockIdx.x = tile, blockIdx.y = job, blockIdx.z strides positions.
__global__ void __launch_bounds__(256)
transpose_kernel(const TransposeJob* __restrict__ jobs, double* __restrict__ trans) {
  __shared__ double tile[32][33];
  const TransposeJob j = jobs[blockIdx.y];
  const int tc = (j.cols + 31) / 32, tr = (j.rows + 31) / 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int pos = blockIdx.z; pos < j.npos; pos += gridDim.z) {
    const double* __restrict__ src = j.src + (int64_t)pos * j.rows * j.cols;
    double* __restrict__ dst = trans + j.dst_off + (int64_t)pos * j.rows * j.cols;
    for (int t = blockIdx.x; t < tr * tc; t += gridDim.x) {
      const int r0 = (t / tc) * 32, c0 = (t % tc) * 32;
      for (int i = ty; i < 32; i += 8) {
        const int r = r0 + i, c = c0 + tx;
        tile[i][tx] = (r < j.rows && c < j.cols) ? src[(int64_t)r * j.cols + c] : 0.0;
      }
      __syncthreads();
      for (int i = ty; i < 32; i += 8) {
        const int c = c0 + i, r = r0 + tx;
        if (c < j.cols && r < j.rows) dst[(int64_t)c * j.rows + r] = tile[tx][i];
      }
      __syncthreads();
    }
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
        v += al * t.A[(int64_t)pos * t.strideA + (int64_t)a * m + a] * t.D[(int64_t)pos * t.strideD + (int64_t)b * p + b];
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

su2_status upload_plan(su2_plan* plan, const std::vector<double>& alpha_host, const std::vector<double>& ident_host,
                       const std::vector<int64_t>& alpha_off_of_task, const std::vector<int64_t>& identA,
                       const std::vector<int64_t>& identD, const std::vector<int64_t>& foldA,
                       const std::vector<int64_t>& foldD, const std::vector<int64_t>& transD, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  int dev = 0;
  SU2_CUDA(cudaGetDevice(&dev));
  SU2_CUDA(cudaDeviceGetAttribute(&plan->num_sms, cudaDevAttrMultiProcessorCount, dev));
  const size_t b_tasks = align256(plan->h_tasks.size() * sizeof(DevTask));
  const size_t b_units = align256(plan->h_units.size() * sizeof(DevUnit));
  const size_t b_work = align256(plan->h_work.size() * sizeof(DevWork));
  const size_t b_red = align256(plan->h_reduce.size() * sizeof(DevReduce));
  const size_t b_diag = align256(plan->h_diag.size() * sizeof(DevDiagTask));
  const size_t b_dbeg = align256(plan->h_diag_begin.size() * sizeof(int32_t));
  const size_t b_psi = align256(plan->psi.size() * sizeof(PsiSector));
  const size_t b_alpha = align256(alpha_host.size() * sizeof(double));
  const size_t b_ident = align256(ident_host.size() * sizeof(double));
  const size_t total = b_tasks + b_units + b_work + b_red + b_diag + b_dbeg + b_psi + b_alpha + b_ident + 256;
  SU2_CUDA(cudaMalloc(&plan->d_blob, total));
  plan->info.plan_device_bytes = (int64_t)total;
  TransposeJob* d_tjobs = nullptr;
  if (plan->trans_elems > 0) {
    bool ok = true;
    for (const TransposeJob& j : plan->h_trans) ok = ok && j.src != nullptr;
    // optional: when the copy does not fit, the tasks keep reading the stored layout
    if (ok && cudaMalloc(&plan->d_trans, (size_t)plan->trans_elems * sizeof(double)) != cudaSuccess) {
      plan->d_trans = nullptr;
      (void)cudaGetLastError();
    }
    if (plan->d_trans) {
      SU2_CUDA(cudaMalloc(&d_tjobs, plan->h_trans.size() * sizeof(TransposeJob)));
      plan->info.plan_device_bytes += plan->trans_elems * (int64_t)sizeof(double);
    }
  }
  FoldJob* d_jobs = nullptr;
  if (plan->fold_elems > 0) {
    SU2_CUDA(cudaMalloc(&plan->d_fold, (size_t)plan->fold_elems * sizeof(double)));
    plan->info.plan_device_bytes += plan->fold_elems * (int64_t)sizeof(double);
    SU2_CUDA(cudaMalloc(&d_jobs, plan->h_fold.size() * sizeof(FoldJob)));
  }
  char* base = (char*)plan->d_blob;
  size_t off = 0;
  auto carve = [&](size_t bytes) { char* p = base + off; off += bytes; return p; };
  plan->d_tasks = (DevTask*)carve(b_tasks);
  plan->d_units = (DevUnit*)carve(b_units);
  plan->d_work = (DevWork*)carve(b_work);
  plan->d_reduce = (DevReduce*)carve(b_red);
  plan->d_diag = (DevDiagTask*)carve(b_diag);
  plan->d_diag_begin = (int32_t*)carve(b_dbeg);
  char* d_psi = carve(b_psi);
  plan->d_alpha = (double*)carve(b_alpha);
  plan->d_identity = (double*)carve(b_ident);
  plan->d_counter = (int32_t*)carve(256);
  // patch device pointers into the host images
  for (size_t i = 0; i < plan->h_tasks.size(); ++i) {
    DevTask& t = plan->h_tasks[i];
    if (alpha_off_of_task[i] >= 0) t.alpha = plan->d_alpha + alpha_off_of_task[i];
    if (identA[i] >= 0) t.A = plan->d_identity + identA[i];
    if (identD[i] >= 0) t.D = plan->d_identity + identD[i];
    if (foldA[i] >= 0) t.A = plan->d_fold + foldA[i];
    if (foldD[i] >= 0) t.D = plan->d_fold + foldD[i];
    if (transD[i] >= 0 && plan->d_trans) {
      t.D = plan->d_trans + transD[i];
      t.flags |= TASK_TRANS_D;
    }
    if (!t.A || !t.D) return SU2_ERR_INVALID_ARGUMENT;   // family without device data
  }
  for (auto& d : plan->h_diag) {
    const DevTask& t = plan->h_tasks[d.pad];
    d.A = t.A; d.D = t.D; d.alpha = t.alpha;
  }
  auto up = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
    if (bytes == 0) return cudaSuccess;
    return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, stream);
  };
  SU2_CUDA(up(plan->d_tasks, plan->h_tasks.data(), plan->h_tasks.size() * sizeof(DevTask)));
  SU2_CUDA(up(plan->d_units, plan->h_units.data(), plan->h_units.size() * sizeof(DevUnit)));
  SU2_CUDA(up(plan->d_work, plan->h_work.data(), plan->h_work.size() * sizeof(DevWork)));
  SU2_CUDA(up(plan->d_reduce, plan->h_reduce.data(), plan->h_reduce.size() * sizeof(DevReduce)));
  SU2_CUDA(up(plan->d_diag, plan->h_diag.data(), plan->h_diag.size() * sizeof(DevDiagTask)));
  SU2_CUDA(up(plan->d_diag_begin, plan->h_diag_begin.data(), plan->h_diag_begin.size() * sizeof(int32_t)));
  SU2_CUDA(up(d_psi, plan->psi.data(), plan->psi.size() * sizeof(PsiSector)));
  SU2_CUDA(up(plan->d_alpha, alpha_host.data(), alpha_host.size() * sizeof(double)));
  SU2_CUDA(up(plan->d_identity, ident_host.data(), ident_host.size() * sizeof(double)));
  if (plan->fold_elems > 0) {
    for (const FoldJob& j : plan->h_fold)
      if (!j.src) { cudaFree(d_jobs); return SU2_ERR_INVALID_ARGUMENT; }   // family without device data
    SU2_CUDA(cudaMemcpyAsync(d_jobs, plan->h_fold.data(), plan->h_fold.size() * sizeof(FoldJob), cudaMemcpyHostToDevice, stream));
    dim3 grid(64, (unsigned)plan->h_fold.size());
    fold_kernel<<<grid, 256, 0, stream>>>(d_jobs, plan->d_alpha, plan->d_fold);
    SU2_CUDA(cudaGetLastError());
    count_launch();
  }
  if (plan->d_trans) {
    SU2_CUDA(cudaMemcpyAsync(d_tjobs, plan->h_trans.data(), plan->h_trans.size() * sizeof(TransposeJob), cudaMemcpyHostToDevice, stream));
    dim3 grid(64, (unsigned)plan->h_trans.size(), 16);
    transpose_kernel<<<grid, 256, 0, stream>>>(d_tjobs, plan->d_trans);
    SU2_CUDA(cudaGetLastError());
    count_launch();
  }
  SU2_CUDA(cudaStreamSynchronize(stream));
  if (d_jobs) cudaFree(d_jobs);
  if (d_tjobs) cudaFree(d_tjobs);
  plan->d_psi_sec = d_psi;
  return SU2_OK;
}

void free_plan_device(su2_plan* plan) {
  if (plan && plan->d_blob) {
    cudaFree(plan->d_blob);
    plan->d_blob = nullptr;
  }
  if (plan && plan->d_fold) {
    cudaFree(plan->d_fold);
    plan->d_fold = nullptr;
  }
  if (plan && plan->d_trans) {
    cudaFree(plan->d_trans);
    plan->d_trans = nullptr;
  }
}

su2_status launch_apply(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  SU2_CUDA(cudaMemsetAsync(plan->d_counter, 0, 8 * sizeof(int32_t), stream));   // [0]: work queue; small plans: one per size class
  su2_status st = plan->small_dm8 > 0 ? launch_heff_small(plan, psi, out, partial, stream_v)
                                      : launch_heff_dmma(plan, psi, out, partial, stream_v);
  if (st != SU2_OK) return st;
  const int nsec = (int)plan->h_reduce.size();
  if (nsec > 0) {
    dim3 grid(32, nsec);
    reduce_kernel<<<grid, 256, 0, stream>>>(plan->d_reduce, partial, out);
    SU2_CUDA(cudaGetLastError());
    count_launch();
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
  if (plan->partial_elems > 0 && !workspace_dev) return SU2_ERR_WORKSPACE;
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
