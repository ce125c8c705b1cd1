// su2_heff_apply_noalloc: H_eff * Psi for callers that cannot allocate device memory (code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc) and so cannot provide the workspace su2_heff_apply wants.
//
// The scratch of the apply -- the partial tiles of the deterministic segmented reduction: one
// partial copy of an output sector per segment, written by the fused GEMM-pair kernel, summed in index order by
// reduce_kernel -- lives in the file-scope device array below instead of a caller-owned workspace.  Everything else is
// the unchanged path: this entry point calls the same launch_apply as su2_heff_apply, so the result is bit-identical.
//
//   * SU2_NOALLOC_SCRATCH_BYTES = 64 MiB is the stated maximum: every GPU that loads the library holds it until the
//     process exits.  It covers BASELINE.json configs[0] and configs[1] (the small-block regime, 37-44 MB of partial
//     tiles); a plan that needs more (configs[2]: 281 MB, configs[3]: 501 MB) is rejected with SU2_ERR_SCRATCH_LIMIT.
//   * In HOST code the array's name is a host-side stand-in, not a device address: handing it to a kernel faults or,
//     where the GPU can reach host memory, silently uses the wrong memory.  The device address is therefore fetched here,
//     in this file, once per device, with that device current, by cudaGetSymbolAddress, and that pointer is what the
//     kernels get.
//   * Nothing in the array has to start at zero: every element of a partial tile that reduce_kernel reads has been
//     written by the fused kernel of the same apply (each (segment, tile) work item stores its whole valid tile), so the
//     contents the previous call left behind are never read.  The array is SHARED by all calls (all plans, all streams)
//     on a device: calls that overlap on the GPU race on it -- order them on one stream, or use su2_heff_apply with
//     private workspaces.
//   * No cudaMalloc, cudaFree, cudaMallocAsync or allocating library routine is called here or below (launch_apply:
//     one cudaMemsetAsync of the plan's queue counter + kernel launches).
#include <cuda_runtime.h>

#include <atomic>
#include <cstdio>
#include <mutex>

#include "su2_internal.h"

namespace {

constexpr size_t SCRATCH_BYTES = (size_t)SU2_NOALLOC_SCRATCH_BYTES;
static __device__ __align__(256) double g_noalloc_scratch[SCRATCH_BYTES / sizeof(double)];

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
std::atomic<double*> g_scratch_ptr[MAX_DEVICES];      // device address of g_noalloc_scratch on device i (null: not yet asked)

// Device address of the scratch array on the CURRENT device (set-up: once per device, with that device current).
su2_status scratch_address(double** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { su2::set_cuda_error("cudaGetDevice", (int)e); return SU2_ERR_CUDA; }
  if (dev < 0 || dev >= MAX_DEVICES) { su2::set_error_text("su2_heff_apply_noalloc: device index beyond 63"); return SU2_ERR_INVALID_ARGUMENT; }
  double* p = g_scratch_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    p = g_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
      e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
      if (e != cudaSuccess || !p) {
        su2::set_cuda_error("cudaGetSymbolAddress(g_noalloc_scratch)", (int)e);
        return SU2_ERR_CUDA;
      }
      g_scratch_ptr[dev].store(p, std::memory_order_release);
    }
  }
  *out = p;
  return SU2_OK;
}

}  // namespace

extern "C" int64_t su2_noalloc_scratch_bytes(void) { return (int64_t)SCRATCH_BYTES; }

extern "C" su2_status su2_heff_apply_noalloc(const su2_plan* plan, const double* psi_dev, double* out_dev, void* cuda_stream) {
  if (!plan || !psi_dev || !out_dev || psi_dev == out_dev) return SU2_ERR_INVALID_ARGUMENT;
  // what launch_apply touches behind the pointer it is given: the fused kernel's partial tiles, or -- two-pass plans -- all of
  // the workspace (the partial slabs of the two-pass route start behind the fused kernel's area)
  const size_t need = plan->tp_partial_elems > 0 ? (size_t)plan->info.workspace_bytes : (size_t)plan->partial_elems * sizeof(double);
  if (need > SCRATCH_BYTES) {
    char buf[256];
    std::snprintf(buf, sizeof(buf),
                  "su2_heff_apply_noalloc: the plan needs %lld bytes of partial tiles, the static scratch holds %lld "
                  "(SU2_NOALLOC_SCRATCH_BYTES); use su2_heff_apply with a caller-owned workspace",
                  (long long)need, (long long)SCRATCH_BYTES);
    su2::set_error_text(buf);
    return SU2_ERR_SCRATCH_LIMIT;
  }
  if (plan->host_only) return SU2_ERR_NO_DEVICE_PLAN;
  double* scratch = nullptr;
  su2_status st = scratch_address(&scratch);
  if (st != SU2_OK) return st;
  return su2::launch_apply(plan, psi_dev, out_dev, scratch, cuda_stream);
}
