// Strided-batched FP64 GEMM-pair microbenchmark entry (BASELINE.json configs[4]):
//   C_b += alpha * A_b X_b B_b^T, one independent item per batch index.
// Implemented as a one-sector-per-item plan-less launch of the same fused kernel path.
#include <cuda_runtime.h>

#include "su2_internal.h"

extern "C" su2_status su2_gemm_pair_batched(int32_t m, int32_t k, int32_t n, int32_t p, int64_t batch, double alpha,
                                            const double* A, const double* X, const double* B, double* C,
                                            void* cuda_stream) {
  if (m <= 0 || k <= 0 || n <= 0 || p <= 0 || batch < 0 || !A || !X || !B || !C) return SU2_ERR_INVALID_ARGUMENT;
  return su2::launch_gemm_pair(m, k, n, p, batch, alpha, A, X, B, C, cuda_stream);
}
