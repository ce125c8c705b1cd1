// Pre-contraction of operator families on the device ("we form pre-contracted
// operators to reduce the N^4 terms to N^2"): a complementary family is a linear combination, over the positions
// (orbital index tuples) of a normal family of the same block, with weights made of the two-electron integrals,
//
//     out[b][pos'][r][c] = sum_pos W[pos'][pos] * in[b][pos][r][c]        for every sector block b of the family.
//
// A block stores its positions contiguously, [npos][rows][ld], so for one block this is ONE row-major
// GEMM  OUT (npos' x E) = W (npos' x npos) . IN (npos x E),  E = rows * ld: the paper's "tall" strided product with
// the position index as the contraction dimension.  FP64 tensor instructions (mma.sync.m8n8k4.f64 = DMMA.8x8x4),
// 64 x 128 output tiles, 8 warps of 32 x 32, cp.async double buffering; operands with 16-byte aligned rows move with
// 16-byte copies.  Sums run over pos in index order inside a thread's accumulator: bit-reproducible.
#include <cuda_runtime.h>

#include <algorithm>

#include "su2_internal.h"

namespace su2 {

namespace {

constexpr int PC_TM = 64, PC_TN = 128, PC_KT = 8, PC_THREADS = 256;
constexpr int PC_LDA = PC_KT + 4;      // 12: A fragments (row g, k t) conflict-free
constexpr int PC_LDB = PC_TN + 4;      // 132: B fragments (k t, column g) conflict-free

__device__ __forceinline__ void pc_cp8(double* dst, const double* src, bool valid) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
  const int sz = valid ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void pc_cp16(double* dst, const double* src, int bytes) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(src), "r"(bytes) : "memory");
}

// C (M x N, ldc) = A (M x K, lda) . B (K x N, ldb), all row-major.  VEC: rows of B are 16-byte aligned.
template <bool VEC>
__global__ void __launch_bounds__(PC_THREADS)
precontract_kernel(int M, int N, int K, const double* __restrict__ A, int lda, const double* __restrict__ B, int64_t ldb,
                   double* __restrict__ C, int64_t ldc) {
  __shared__ __align__(16) double As[2][PC_TM * PC_LDA];
  __shared__ __align__(16) double Bs[2][PC_KT * PC_LDB];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, t = lane & 3;
  const int wm = warp >> 2, wn = warp & 3;                      // 2 x 4 warps, 32 x 32 each
  const int m0 = blockIdx.y * PC_TM;
  const int64_t n0 = (int64_t)blockIdx.x * PC_TN;

  auto stage = [&](int buf, int k0) {
    // A tile: 64 rows x 16 k (8-byte copies, zero fill outside)
    for (int e = tid; e < PC_TM * PC_KT; e += PC_THREADS) {
      const int r = e / PC_KT, kk = e % PC_KT;
      const bool ok = m0 + r < M && k0 + kk < K;
      pc_cp8(&As[buf][r * PC_LDA + kk], ok ? A + (int64_t)(m0 + r) * lda + k0 + kk : A, ok);
    }
    // B tile: 16 k x 128 columns
    if (VEC) {
      for (int e = tid; e < PC_KT * (PC_TN / 2); e += PC_THREADS) {
        const int kk = e / (PC_TN / 2), c = 2 * (e % (PC_TN / 2));
        const int64_t col = n0 + c;
        int bytes = 0;
        if (k0 + kk < K && col < N) bytes = col + 1 < N ? 16 : 8;
        pc_cp16(&Bs[buf][kk * PC_LDB + c], bytes ? B + (int64_t)(k0 + kk) * ldb + col : B, bytes);
      }
    } else {
      for (int e = tid; e < PC_KT * PC_TN; e += PC_THREADS) {
        const int kk = e / PC_TN, c = e % PC_TN;
        const bool ok = k0 + kk < K && n0 + c < N;
        pc_cp8(&Bs[buf][kk * PC_LDB + c], ok ? B + (int64_t)(k0 + kk) * ldb + n0 + c : B, ok);
      }
    }
    asm volatile("cp.async.commit_group;\n" ::: "memory");
  };

  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  const int nk = (K + PC_KT - 1) / PC_KT;
  stage(0, 0);
  for (int s = 0; s < nk; ++s) {
    if (s + 1 < nk) {
      stage((s + 1) & 1, (s + 1) * PC_KT);
      asm volatile("cp.async.wait_group 1;\n" ::: "memory");
    } else {
      asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    }
    __syncthreads();
    const double* a = &As[s & 1][(wm * 32 + g) * PC_LDA + t];
    const double* b = &Bs[s & 1][t * PC_LDB + wn * 32 + g];
#pragma unroll
    for (int sub = 0; sub < PC_KT / 4; ++sub) {
      double af[4], bf[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) af[i] = a[i * 8 * PC_LDA + sub * 4];
#pragma unroll
      for (int j = 0; j < 4; ++j) bf[j] = b[sub * 4 * PC_LDB + j * 8];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
          asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
              : "+d"(acc[i][j][0]), "+d"(acc[i][j][1])
              : "d"(af[i]), "d"(bf[j]));
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int r = m0 + wm * 32 + i * 8 + g;
      const int64_t c = n0 + wn * 32 + j * 8 + 2 * t;
      if (r < M) {
        double* o = C + (int64_t)r * ldc + c;
        if (c < N) o[0] = acc[i][j][0];
        if (c + 1 < N) o[1] = acc[i][j][1];
      }
    }
}

}  // namespace

}  // namespace su2

using namespace su2;

extern "C" su2_status su2_precontract(int32_t nblk, const int64_t* block_elems, const int64_t* in_off, const int64_t* out_off,
                                      int32_t npos_in, int32_t npos_out, const double* w_dev, const double* in_dev,
                                      double* out_dev, void* cuda_stream) {
  if (nblk < 0 || npos_in <= 0 || npos_out <= 0 || !w_dev || !in_dev || !out_dev || in_dev == out_dev) return SU2_ERR_INVALID_ARGUMENT;
  if (nblk > 0 && (!block_elems || !in_off || !out_off)) return SU2_ERR_INVALID_ARGUMENT;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  for (int b = 0; b < nblk; ++b) {
    const int64_t e = block_elems[b];
    if (e < 0 || in_off[b] < 0 || out_off[b] < 0) return SU2_ERR_INVALID_ARGUMENT;
    if (e == 0) continue;
    const double* in = in_dev + in_off[b];
    double* out = out_dev + out_off[b];
    const int64_t ntile = (e + PC_TN - 1) / PC_TN;
    if (ntile > 2147483647LL) return SU2_ERR_INVALID_ARGUMENT;
    dim3 grid((unsigned)ntile, (unsigned)((npos_out + PC_TM - 1) / PC_TM));
    const bool vec = !(e & 1) && !((uintptr_t)in & 15);
    if (vec) precontract_kernel<true><<<grid, PC_THREADS, 0, stream>>>(npos_out, (int)std::min<int64_t>(e, 2147483647LL), npos_in, w_dev, npos_in, in, e, out, e);
    else precontract_kernel<false><<<grid, PC_THREADS, 0, stream>>>(npos_out, (int)std::min<int64_t>(e, 2147483647LL), npos_in, w_dev, npos_in, in, e, out, e);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) { set_cuda_error("precontract_kernel launch", (int)err); return SU2_ERR_CUDA; }
    count_launch();
  }
  return SU2_OK;
}
