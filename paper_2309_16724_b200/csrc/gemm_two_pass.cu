// The strided-batched GEMM pair in its UN-FUSED form (route 4 of su2_gemm_pair_batched_route; BASELINE.json configs[4],
// PAPER.md:116-136): pass 1 writes T_b = alpha A_b X_b (or alpha X_b B_b^T, whichever order is cheaper) to a stream-ordered
// scratch, pass 2 forms C_b += T_b B_b^T (or A_b T_b).
//
// Both passes run on tp_gemm_kernel (heff_two_pass.cu), the kernel of the apply's two-pass route: the batch items take the place
// of the positions of ONE task (A_b, B_b = the operator blocks of position b), with two differences expressed as slice flags --
// every item has its own X_b (third coordinate of the E map = item) and its own output, which pass 2 accumulates into directly
// (chunk = 1, accumulators initialised from C_b).  Why un-fused: on sm_100a what decides DMMA throughput is the register tile of
// a warp and the number of independent CTAs per SM (profiles/r02_cfg5_shapes.md); 64 x 128 CTA tiles with four warps of 32 x 64
// and two CTAs per SM reach 90-95 % of the pipe, the fused kernel 79 %.  Ragged outputs run narrower edge tiles, and a CTA works
// through several consecutive (item, tile) pairs with its pipeline kept full, so short inner extents (128) do not pay a CTA
// start-up per tile.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <mutex>

#include "su2_internal.h"

namespace su2 {

namespace {
// The scratch comes from a memory pool of this library's own: the device's default pool hands freed memory back to the driver at
// the next synchronisation, so a caller that synchronises between calls would pay a fresh allocation of hundreds of MB every
// call (measured: 2.6 ms per call, more than the two passes of 178 items of 512^4).  This pool keeps up to 2 GiB across
// synchronisations; what a call needs beyond that is still returned.
std::mutex g_pool_mutex;
cudaMemPool_t g_pool[64] = {};
su2_status scratch_pool(cudaMemPool_t* out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= 64) { set_cuda_error("cudaGetDevice", (int)e); return SU2_ERR_CUDA; }
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  if (!g_pool[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t pool;
    e = cudaMemPoolCreate(&pool, &props);
    if (e != cudaSuccess) { set_cuda_error("cudaMemPoolCreate", (int)e); return SU2_ERR_CUDA; }
    uint64_t keep = (uint64_t)2 << 30;
    e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    if (e != cudaSuccess) { set_cuda_error("cudaMemPoolSetAttribute", (int)e); return SU2_ERR_CUDA; }
    g_pool[dev] = pool;
  }
  *out = g_pool[dev];
  return SU2_OK;
}
}  // namespace

// stream-ordered allocation from that pool (freed with cudaFreeAsync)
su2_status gemm_scratch_alloc(void** out, size_t bytes, void* stream_v) {
  cudaMemPool_t pool;
  su2_status st = scratch_pool(&pool);
  if (st != SU2_OK) return st;
  cudaError_t e = cudaMallocFromPoolAsync(out, bytes, pool, (cudaStream_t)stream_v);
  if (e != cudaSuccess) { set_cuda_error("cudaMallocFromPoolAsync(gemm_pair scratch)", (int)e); return SU2_ERR_CUDA; }
  return SU2_OK;
}

// C_b += alpha (A_b X_b) B_b^T in two passes; operands with even leading dimensions and 16-byte aligned bases (the caller
// re-pitches the others); T and the three small tables live in stream-ordered allocations.
su2_status launch_gemm_two_pass(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, int ldA, const double* X, int ldX,
                                const double* B, int ldB, double* C, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  const bool o1 = 2.0 * m * k * n + 2.0 * m * n * p > 2.0 * k * n * p + 2.0 * m * k * p;   // X B^T first is cheaper
  const int rowsT = o1 ? k : m, colsT = o1 ? p : n, ldt = (colsT + 3) & ~3;
  const int K1 = o1 ? n : k, K2 = o1 ? k : n;
  const int64_t tiles1 = (int64_t)((rowsT + TP_TM - 1) / TP_TM) * ((colsT + TP_TN - 1) / TP_TN);
  const int64_t tiles2 = (int64_t)((m + TP_TM - 1) / TP_TM) * ((p + TP_TN - 1) / TP_TN);
  // items per launch: 32-bit item numbers and row coordinates, and a scratch of at most 8 GiB
  const int64_t per_item = (int64_t)rowsT * ldt;
  int64_t nb_max = std::min<int64_t>({batch, ((int64_t)1 << 30) / std::max(tiles1, tiles2), ((int64_t)1 << 30) / rowsT,
                                      std::max<int64_t>(1, ((int64_t)1 << 30) / per_item)});
  struct Tables {
    alignas(128) unsigned char maps[4 * 128];
    DevTask task;
    TpSlice slice;
  };
  char* dev = nullptr;
  cudaMemPool_t pool;
  su2_status st = scratch_pool(&pool);
  if (st != SU2_OK) return st;
  cudaError_t e = cudaMallocFromPoolAsync((void**)&dev, sizeof(Tables) + 256 + (size_t)nb_max * per_item * sizeof(double), pool, stream);
  if (e != cudaSuccess) { set_cuda_error("cudaMallocAsync(gemm_two_pass T)", (int)e); return SU2_ERR_CUDA; }
  double* T = (double*)(dev + ((sizeof(Tables) + 255) & ~(size_t)255));
  for (int64_t b0 = 0; b0 < batch && st == SU2_OK; b0 += nb_max) {
    const int nb = (int)std::min<int64_t>(nb_max, batch - b0);
    const double *Ab = A + b0 * m * (int64_t)ldA, *Xb = X + b0 * k * (int64_t)ldX, *Bb = B + b0 * p * (int64_t)ldB;
    Tables h;
    std::memset(&h, 0, sizeof(h));
    if ((st = encode_tensor_map(h.maps + 0, MapKey{Ab, m, k, ldA, nb, (int64_t)m * ldA, TP_KS, TP_TM})) != SU2_OK) break;       // A: left, as stored
    if ((st = encode_tensor_map(h.maps + 128, MapKey{Bb, p, n, ldB, nb, (int64_t)p * ldB, TP_KS, TP_TN})) != SU2_OK) break;     // B^T: right, inner index contiguous
    if ((st = encode_tensor_map(h.maps + 256, MapKey{Xb, k, n, ldX, nb, (int64_t)k * ldX, o1 ? TP_KS : TP_RLD, o1 ? TP_TM : TP_KS})) != SU2_OK) break;
    if ((st = encode_tensor_map(h.maps + 384, MapKey{T, (int32_t)((int64_t)nb * rowsT), colsT, ldt, 1, (int64_t)nb * rowsT * ldt,
                                                     o1 ? TP_RLD : TP_KS, o1 ? TP_KS : TP_TM})) != SU2_OK) break;
    DevTask& t = h.task;
    t.A = Ab; t.D = Bb; t.alpha = nullptr; t.coef = alpha;
    t.m = m; t.k = k; t.n = n; t.p = p; t.strideA = m * ldA; t.strideD = p * ldB; t.ldA = ldA; t.ldD = ldB; t.npos = nb; t.flags = 0;
    TpSlice& sl = h.slice;
    sl.task = 0; sl.pos0 = 0; sl.npos = nb; sl.order = o1 ? 1 : 0; sl.t_row0 = 0; sl.ldt = ldt;
    sl.mapA = 0; sl.mapD = 1; sl.mapE = 2; sl.mapT = 3; sl.item1 = 0; sl.item2 = 0; sl.chunk = 1; sl.nchunk = nb; sl.part_off = 0;
    sl.flags = TP_SLICE_E_PER_POS | TP_SLICE_ACCUMULATE;
    e = cudaMemcpyAsync(dev, &h, sizeof(h), cudaMemcpyHostToDevice, stream);   // pageable source: staged before the call returns
    if (e != cudaSuccess) { set_cuda_error("cudaMemcpyAsync(gemm_two_pass tables)", (int)e); st = SU2_ERR_CUDA; break; }
    const Tables* d = (const Tables*)dev;
    // consecutive items per CTA: an inner loop of about 2048 per CTA, at least ~8 waves of CTAs
    auto ipc_for = [](int K, int64_t items) {
      int64_t ipc = (int64_t)std::lround(2048.0 / K);
      ipc = std::min<int64_t>(ipc, items / (8 * 296));
      return (int)std::max<int64_t>(1, std::min<int64_t>(ipc, 64));
    };
    const int64_t items1 = tiles1 * nb, items2 = tiles2 * nb;
    st = launch_tp_gemm(&d->slice, 1, 0, (int)items1, ipc_for(K1, items1), &d->task, d->maps, T, C + b0 * m * (int64_t)p, stream_v);
    if (st == SU2_OK)
      st = launch_tp_gemm(&d->slice, 1, 1, (int)items2, ipc_for(K2, items2), &d->task, d->maps, T, C + b0 * m * (int64_t)p, stream_v);
  }
  cudaFreeAsync(dev, stream);
  return st;
}

}  // namespace su2
