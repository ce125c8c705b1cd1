// The strided-batched GEMM pair in its UN-FUSED form (route 4 of su2_gemm_pair_batched_route; BASELINE.json configs[4],
// PAPER.md:116-136): pass 1 writes T_b = A_b X_b to a stream-ordered scratch, pass 2 adds alpha T_b B_b^T to C_b.
//
// Why it exists next to the fused kernel (heff_tma.cu): on sm_100a the FP64 tensor instruction is DMMA.8x8x4 and what decides
// its throughput is the register tile of a warp and how many independent CTAs an SM holds (profiles/r02_cfg5_shapes.md: the
// vendor GEMM reaches 96 % of the pipe with four warps of 32 x 64 tiles and two CTAs per SM).  The fused kernel keeps both
// products' accumulators in registers and the T chunk in shared memory, which pins it to 12 warps of 32 x 48 / 32 x 16 tiles in
// one CTA per SM (78 %).  For items of >= 128 the round trip of T through L2 / HBM (16 bytes per entry against >= 500 flops)
// costs less than that.  One kernel serves both passes:
//
//   D_b (M x N) = beta D_b + alpha L_b (M x K) R_b,   R_b given as K x N (N contiguous: X as stored) or N x K (K contiguous: B)
//
// CTA = one producer warp (one elected thread issues every bulk-tensor copy) + four consumer warps (2 x 2, each 32 x 64: 64
// accumulator doubles, 32 DMMAs per 12 fragment loads and k4 step); CTA tile 64 x 128, stages of 20 k (box pitches = 4 mod 8
// doubles: conflict-free fragment loads without swizzling), 3 stages = 92 KB, two CTAs per SM.  Ragged extents: the tensor maps
// carry the true extents (out-of-bounds elements arrive as zeros), the epilogue is guarded.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "su2_internal.h"

namespace su2 {

namespace {

constexpr int G_TM = 64, G_TN = 128, G_KS = 20, G_NS = 3;
constexpr int G_CONSUMERS = 4, G_THREADS = 32 * (G_CONSUMERS + 1);
constexpr int G_LBOX = G_TM * G_KS;                       // L box: 64 rows x 20 k (pitch 20)
constexpr int G_RBOX_K = G_TN * G_KS;                     // R box, K-major: 128 rows x 20 k (pitch 20)
constexpr int G_RLD = G_TN + 4;                           // R box, N-major: 20 k-rows x 132 columns (pitch 132)
constexpr int G_RBOX_N = G_KS * G_RLD;
constexpr int G_RBOX = G_RBOX_N > G_RBOX_K ? G_RBOX_N : G_RBOX_K;
constexpr int G_STAGE = G_LBOX + G_RBOX;                  // doubles per stage
static_assert(G_LBOX % 16 == 0 && G_STAGE % 16 == 0, "boxes land on 128-byte boundaries");
constexpr size_t G_SMEM = (size_t)G_NS * G_STAGE * sizeof(double);

__device__ __forceinline__ unsigned g_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void g_mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(g_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void g_mbar_arrive(uint64_t* bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(g_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void g_mbar_expect(uint64_t* bar, unsigned bytes) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"(g_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void g_mbar_wait(uint64_t* bar, int parity) {
  unsigned ok = 0;
  while (!ok)
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(ok) : "r"(g_smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void g_tma_box(unsigned dst, const void* map, int c0, int c1, int c2, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n"
               ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(g_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void g_dmma(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// maps[0]: L {K, M, batch} box {20, 64};  maps[1]: R, either {K, N, batch} box {20, 128} or (R_NMAJOR) {N, K, batch} box {132, 20}
template <bool R_NMAJOR>
__global__ void __launch_bounds__(G_THREADS, 2)
dgemm_tma_kernel(const __grid_constant__ CUtensorMap mapL, const __grid_constant__ CUtensorMap mapR, int M, int N, int K,
                 double alpha, double beta, double* __restrict__ D, int64_t strideD, int ldd) {
  extern __shared__ __align__(1024) double smem[];
  __shared__ __align__(8) uint64_t full[G_NS];
  __shared__ __align__(8) uint64_t empty[G_NS];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int row0 = blockIdx.y * G_TM, col0 = blockIdx.x * G_TN, item = blockIdx.z;
  const int nsteps = (K + G_KS - 1) / G_KS;
  if (tid == 0) {
    for (int i = 0; i < G_NS; ++i) {
      g_mbar_init(&full[i], 1);
      g_mbar_init(&empty[i], G_CONSUMERS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  if (warp == G_CONSUMERS) {
    // ---- producer: one thread, two boxes per stage
    if (lane != 0) return;
    constexpr unsigned bytes = (unsigned)((G_LBOX + (R_NMAJOR ? G_RBOX_N : G_RBOX_K)) * sizeof(double));
    for (int s = 0; s < nsteps; ++s) {
      const int b = s % G_NS, round = s / G_NS;
      if (round > 0) g_mbar_wait(&empty[b], (round - 1) & 1);
      g_mbar_expect(&full[b], bytes);
      const unsigned st = g_smem_u32(smem + (size_t)b * G_STAGE);
      g_tma_box(st, &mapL, s * G_KS, row0, item, &full[b]);
      if (R_NMAJOR) g_tma_box(st + G_LBOX * 8u, &mapR, col0, s * G_KS, item, &full[b]);
      else g_tma_box(st + G_LBOX * 8u, &mapR, s * G_KS, col0, item, &full[b]);
    }
    return;
  }
  // ---- consumers: warp (wr, wc) of a 2 x 2 grid owns rows [32 wr, +32) x columns [64 wc, +64) of the tile
  const int wr = warp >> 1, wc = warp & 1;
  const int g = lane >> 2, t = lane & 3;
  double acc[4][8][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  const int l_off = (wr * 32 + g) * G_KS + t;                                   // L[row][k]
  const int r_off = G_LBOX + (R_NMAJOR ? t * G_RLD + wc * 64 + g : (wc * 64 + g) * G_KS + t);
  for (int s = 0; s < nsteps; ++s) {
    const int b = s % G_NS;
    g_mbar_wait(&full[b], (s / G_NS) & 1);
    const double* __restrict__ st = smem + (size_t)b * G_STAGE;
    // fragments of sub-step s + 1 are fetched into a second register set before the 32 DMMAs of sub-step s are issued
    double af[2][4], bf[2][8];
#pragma unroll
    for (int i = 0; i < 4; ++i) af[0][i] = st[l_off + i * 8 * G_KS];
#pragma unroll
    for (int j = 0; j < 8; ++j) bf[0][j] = st[r_off + (R_NMAJOR ? j * 8 : j * 8 * G_KS)];
#pragma unroll
    for (int sub = 0; sub < G_KS / 4; ++sub) {
      const int cur = sub & 1, nxt = cur ^ 1;
      if (sub + 1 < G_KS / 4) {
#pragma unroll
        for (int i = 0; i < 4; ++i) af[nxt][i] = st[l_off + i * 8 * G_KS + (sub + 1) * 4];
#pragma unroll
        for (int j = 0; j < 8; ++j) bf[nxt][j] = st[r_off + (R_NMAJOR ? (sub + 1) * 4 * G_RLD + j * 8 : j * 8 * G_KS + (sub + 1) * 4)];
      }
#pragma unroll
      for (int j = 0; j < 8; ++j)
#pragma unroll
        for (int i = 0; i < 4; ++i) g_dmma(acc[i][j], af[cur][i], bf[cur][j]);
    }
    __syncwarp();
    if (lane == 0) g_mbar_arrive(&empty[b]);
  }
  // ---- epilogue: D = beta D + alpha acc (accumulator layout: row g, columns 2t, 2t + 1 of every m8n8 tile).  With beta != 0
  // all old values are fetched first (32 independent 16-byte loads in flight), then combined and stored: fetching them one by
  // one in front of each store cost 14 % of the second pass at 512^4
  double* __restrict__ dst = D + (int64_t)item * strideD;
  const bool vec = !(ldd & 1);
  const int cbase = col0 + wc * 64 + 2 * t;
  if (beta != 0.0) {
    double2 old[4][8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = row0 + wr * 32 + i * 8 + g;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int c = cbase + j * 8;
        const double* o = dst + (int64_t)r * ldd + c;
        old[i][j] = make_double2(0.0, 0.0);
        if (r < M) {
          if (vec && c + 1 < N) old[i][j] = *(const double2*)o;
          else {
            if (c < N) old[i][j].x = o[0];
            if (c + 1 < N) old[i][j].y = o[1];
          }
        }
      }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        acc[i][j][0] = beta * old[i][j].x + alpha * acc[i][j][0];
        acc[i][j][1] = beta * old[i][j].y + alpha * acc[i][j][1];
      }
  } else {
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) { acc[i][j][0] *= alpha; acc[i][j][1] *= alpha; }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = row0 + wr * 32 + i * 8 + g;
    if (r >= M) continue;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int c = cbase + j * 8;
      double* o = dst + (int64_t)r * ldd + c;
      if (vec && c + 1 < N) *(double2*)o = make_double2(acc[i][j][0], acc[i][j][1]);
      else {
        if (c < N) o[0] = acc[i][j][0];
        if (c + 1 < N) o[1] = acc[i][j][1];
      }
    }
  }
}

template <bool R_NMAJOR>
su2_status launch_dgemm(const void* L, int ldl, int64_t strideL, const void* R, int ldr, int64_t strideR, int M, int N, int K, int batch,
                        double alpha, double beta, double* D, int64_t strideD, int ldd, cudaStream_t stream) {
  static bool attr_done[64] = {};
  int dev = 0;
  cudaGetDevice(&dev);
  if (!attr_done[dev & 63]) {
    cudaError_t e = cudaFuncSetAttribute(dgemm_tma_kernel<R_NMAJOR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G_SMEM);
    if (e != cudaSuccess) { set_cuda_error("cudaFuncSetAttribute(dgemm_tma_kernel)", (int)e); return SU2_ERR_CUDA; }
    attr_done[dev & 63] = true;
  }
  alignas(64) CUtensorMap mapL, mapR;
  su2_status st;
  if ((st = encode_tensor_map(&mapL, MapKey{L, M, K, ldl, batch, strideL, G_KS, G_TM})) != SU2_OK) return st;
  if (R_NMAJOR) st = encode_tensor_map(&mapR, MapKey{R, K, N, ldr, batch, strideR, G_RLD, G_KS});
  else st = encode_tensor_map(&mapR, MapKey{R, N, K, ldr, batch, strideR, G_KS, G_TN});
  if (st != SU2_OK) return st;
  dim3 grid((N + G_TN - 1) / G_TN, (M + G_TM - 1) / G_TM, batch);
  dgemm_tma_kernel<R_NMAJOR><<<grid, G_THREADS, G_SMEM, stream>>>(mapL, mapR, M, N, K, alpha, beta, D, strideD, ldd);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_cuda_error("dgemm_tma_kernel launch", (int)e); return SU2_ERR_CUDA; }
  count_launch();
  return SU2_OK;
}

}  // namespace

// C_b += alpha (A_b X_b) B_b^T in two passes; operands with even leading dimensions and 16-byte aligned bases (the caller
// re-pitches the others); T lives in a stream-ordered allocation of batch * m * ldt doubles.
su2_status launch_gemm_two_pass(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, int ldA, const double* X, int ldX,
                                const double* B, int ldB, double* C, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  if (batch > 65535) return SU2_ERR_INVALID_ARGUMENT;         // grid.z
  const int ldt = n + (n & 1);
  double* T = nullptr;
  cudaError_t e = cudaMallocAsync((void**)&T, (size_t)batch * m * ldt * sizeof(double), stream);
  if (e != cudaSuccess) { set_cuda_error("cudaMallocAsync(gemm_two_pass T)", (int)e); return SU2_ERR_CUDA; }
  su2_status st = launch_dgemm<true>(A, ldA, (int64_t)m * ldA, X, ldX, (int64_t)k * ldX, m, n, k, (int)batch, 1.0, 0.0, T, (int64_t)m * ldt, ldt, stream);
  if (st == SU2_OK)
    st = launch_dgemm<false>(T, ldt, (int64_t)m * ldt, B, ldB, (int64_t)p * ldB, m, p, n, (int)batch, alpha, 1.0, C, (int64_t)m * p, p, stream);
  cudaFreeAsync(T, stream);
  return st;
}

}  // namespace su2
