// Small-block regime of the strided-batched FP64 GEMM pair (BASELINE.json configs[4]; the paper's
// "strided batched matrix multiplication" sequences, for blocks of a few doubles to a few
// dozen doubles):  C_b += alpha * A_b (m x k) X_b (k x n) B_b^T (n x p), one independent item per batch index.
//
// At these sizes the item is HBM-bound (8 (mk + kn + pn + 2mp) bytes against 2mkn + 2mnp flops: b/10 flop/B
// for square b), so the kernel is built around memory-level parallelism, not around the FP64 pipe:
//   * one CTA of WPI warps (1 to 16, one per 16 x 16 macro tile) per item at a time, many CTAs per SM (shared
//     memory is sized by the actual item shape: 2.5 KB at b = 8, 215 KB at b = 80), persistent over the batch
//     with a grid-stride loop;
//   * A, X and B move global -> shared with cp.async (16-byte when rows allow it, else 8-byte), no register
//     staging; with NBUF = 2 the copies of the NEXT item are in flight while the current one is multiplied;
//     the C lines of the item are prefetched into L2 at the same time;
//   * both products run on DMMA.8x8x4 (mma.sync.m8n8k4.f64) out of shared memory, rows padded to a stride
//     = 4 (mod 8) doubles so fragment loads are bank-conflict free; T = A X goes through shared memory only;
//   * pad rows/columns of the shared tiles are zeroed once per CTA (every item of a call has the same shape, so
//     the copies never touch them) -- ragged shapes cost nothing but the round-up to 8 (4 along k).
// Deterministic: one CTA owns an item, no atomics.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "su2_internal.h"

namespace su2 {

namespace {

__host__ __device__ inline int ru(int x, int q) { return (x + q - 1) / q * q; }
// leading dimension >= x with ld = 4 (mod 8): DMMA fragment loads (8 rows x 4 consecutive doubles per
// half-warp) then hit 16 distinct 8-byte banks
__host__ __device__ inline int ld_of(int x) { return ((x + 3) & ~7) + 4; }

struct SmallGeom {
  int M8, K4, N8, P8;        // padded extents
  int ldA, ldX, ldB, ldT;    // leading dimensions in shared memory (doubles)
  int szA, szX, szB, szT;    // tile sizes (doubles)
};

__host__ __device__ inline SmallGeom small_geom(int m, int k, int n, int p) {
  SmallGeom g;
  g.M8 = ru(m, 8); g.K4 = ru(k, 4); g.N8 = ru(n, 8); g.P8 = ru(p, 8);
  g.ldA = ld_of(g.K4); g.ldX = ld_of(g.N8); g.ldB = ld_of(g.N8); g.ldT = ld_of(g.N8);
  g.szA = g.M8 * g.ldA; g.szX = g.K4 * g.ldX; g.szB = g.P8 * g.ldB; g.szT = g.M8 * g.ldT;
  return g;
}

__device__ __forceinline__ void cp_async8(double* dst, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async16(double* dst, const double* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// dense row-major rows x cols (contiguous) -> shared tile with leading dimension ld; VEC doubles per copy.
// (r, c) advance incrementally: no division inside the loop.
template <int VEC>
__device__ __forceinline__ void copy_tile(double* __restrict__ dst, int ld, const double* __restrict__ src, int rows, int cols,
                                          int tid, int nthr) {
  const int cv = cols / VEC;                 // copies per row
  const int total = rows * cv;
  int r = tid / cv, c = tid - r * cv;
  const int dr = nthr / cv, dc = nthr - dr * cv;
  for (int e = tid; e < total; e += nthr) {
    if (VEC == 2) cp_async16(dst + r * ld + 2 * c, src + (int64_t)r * cols + 2 * c);
    else cp_async8(dst + r * ld + c, src + (int64_t)r * cols + c);
    r += dr; c += dc;
    if (c >= cv) { c -= cv; ++r; }
  }
}

template <int WPI>
__device__ __forceinline__ void group_sync() {
  if (WPI == 1) __syncwarp(); else __syncthreads();
}

}  // namespace

// CTA = WPI warps; items blockIdx.x, blockIdx.x + gridDim.x, ...
template <int WPI>
__global__ void __launch_bounds__(32 * WPI)
gemm_pair_small_kernel(int m, int k, int n, int p, int64_t batch, double alpha, const double* __restrict__ A,
                       const double* __restrict__ X, const double* __restrict__ B, double* __restrict__ C, int nbuf,
                       int vec_ok) {
  extern __shared__ __align__(16) double smem[];
  const SmallGeom g = small_geom(m, k, n, p);
  const int tid = threadIdx.x, nthr = 32 * WPI, lane = tid & 31, warp = tid >> 5;
  const int in_sz = g.szA + g.szX + g.szB;         // one input buffer set
  double* const Ts = smem + nbuf * in_sz;
  // zero everything once: pad rows / columns are never written again
  for (int e = tid; e < nbuf * in_sz + g.szT; e += nthr) smem[e] = 0.0;
  group_sync<WPI>();

  const int64_t szA = (int64_t)m * k, szX = (int64_t)k * n, szB = (int64_t)p * n, szC = (int64_t)m * p;
  auto issue = [&](int64_t b, int buf) {
    double* As = smem + buf * in_sz;
    double* Xs = As + g.szA;
    double* Bs = Xs + g.szX;
    if (vec_ok) {
      copy_tile<2>(As, g.ldA, A + b * szA, m, k, tid, nthr);
      copy_tile<2>(Xs, g.ldX, X + b * szX, k, n, tid, nthr);
      copy_tile<2>(Bs, g.ldB, B + b * szB, p, n, tid, nthr);
    } else {
      copy_tile<1>(As, g.ldA, A + b * szA, m, k, tid, nthr);
      copy_tile<1>(Xs, g.ldX, X + b * szX, k, n, tid, nthr);
      copy_tile<1>(Bs, g.ldB, B + b * szB, p, n, tid, nthr);
    }
    // the item's C lines: read late, so pull them into L2 now
    const double* c0 = C + b * szC;
    for (int64_t e = (int64_t)tid * 16; e < szC; e += (int64_t)nthr * 16)
      asm volatile("prefetch.global.L2 [%0];\n" ::"l"(c0 + e));
  };

  const int mt = g.M8 / 8, nt = g.N8 / 8, pt = g.P8 / 8;
  const int mm = (mt + 1) / 2, nn = (nt + 1) / 2, pp = (pt + 1) / 2;   // 16 x 16 macro tiles
  const int fr = lane >> 2, fc = lane & 3;                              // fragment row / column of this lane

  int64_t b = blockIdx.x;
  if (nbuf == 2) {
    if (b < batch) issue(b, 0);
    cp_async_commit();
  }
  for (int it = 0; b < batch; b += gridDim.x, ++it) {
    const int buf = (nbuf == 2) ? (it & 1) : 0;
    if (nbuf == 2) {
      if (b + gridDim.x < batch) issue(b + gridDim.x, buf ^ 1);
      cp_async_commit();
      cp_async_wait<1>();
    } else {
      issue(b, 0);
      cp_async_commit();
      cp_async_wait<0>();
    }
    group_sync<WPI>();
    const double* As = smem + buf * in_sz;
    const double* Xs = As + g.szA;
    const double* Bs = Xs + g.szX;

    // ---- first product: T = A X, macro tiles round-robin over the warps
    for (int t = warp; t < mm * nn; t += WPI) {
      const int r0 = (t / nn) * 16, c0 = (t % nn) * 16;
      const bool r1 = r0 + 8 < g.M8, c1 = c0 + 8 < g.N8;          // warp-uniform
      double acc[2][2][2] = {};
      const double* a0p = As + (r0 + fr) * g.ldA + fc;
      const double* a1p = a0p + (r1 ? 8 * g.ldA : 0);
      const double* x0p = Xs + fc * g.ldX + c0 + fr;
      const double* x1p = x0p + (c1 ? 8 : 0);
#pragma unroll 2
      for (int k0 = 0; k0 < g.K4; k0 += 4) {
        const double a0 = a0p[k0], a1 = a1p[k0];
        const double x0 = x0p[k0 * g.ldX], x1 = x1p[k0 * g.ldX];
        dmma(acc[0][0], a0, x0);
        if (c1) dmma(acc[0][1], a0, x1);
        if (r1) dmma(acc[1][0], a1, x0);
        if (r1 && c1) dmma(acc[1][1], a1, x1);
      }
#pragma unroll
      for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
          if ((i == 0 || r1) && (j == 0 || c1))
            *reinterpret_cast<double2*>(Ts + (r0 + 8 * i + fr) * g.ldT + c0 + 8 * j + 2 * fc) = make_double2(acc[i][j][0], acc[i][j][1]);
    }
    group_sync<WPI>();

    // ---- second product: C += alpha T B^T
    double* __restrict__ Cb = C + b * szC;
    for (int t = warp; t < mm * pp; t += WPI) {
      const int r0 = (t / pp) * 16, c0 = (t % pp) * 16;
      const bool r1 = r0 + 8 < g.M8, c1 = c0 + 8 < g.P8;
      double acc[2][2][2] = {};
      const double* t0p = Ts + (r0 + fr) * g.ldT + fc;
      const double* t1p = t0p + (r1 ? 8 * g.ldT : 0);
      const double* b0p = Bs + (c0 + fr) * g.ldB + fc;
      const double* b1p = b0p + (c1 ? 8 * g.ldB : 0);
#pragma unroll 2
      for (int k0 = 0; k0 < g.N8; k0 += 4) {
        const double a0 = t0p[k0], a1 = t1p[k0];
        const double x0 = b0p[k0], x1 = b1p[k0];
        dmma(acc[0][0], a0, x0);
        if (c1) dmma(acc[0][1], a0, x1);
        if (r1) dmma(acc[1][0], a1, x0);
        if (r1 && c1) dmma(acc[1][1], a1, x1);
      }
#pragma unroll
      for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const int r = r0 + 8 * i + fr, c = c0 + 8 * j + 2 * fc;
          if (r < m) {
            double* dst = Cb + (int64_t)r * p + c;
            if (vec_ok && c + 1 < p) {                  // p even and C 16-byte aligned
              double2 v = *reinterpret_cast<double2*>(dst);
              v.x += alpha * acc[i][j][0]; v.y += alpha * acc[i][j][1];
              *reinterpret_cast<double2*>(dst) = v;
            } else {
              if (c < p) dst[0] += alpha * acc[i][j][0];
              if (c + 1 < p) dst[1] += alpha * acc[i][j][1];
            }
          }
        }
    }
    group_sync<WPI>();       // Ts and this input buffer are free again
  }
  cp_async_wait<0>();
}

// Shared memory (bytes) of one CTA; the router in gemm_pair.cu uses it to decide whether an item shape
// belongs to the small-block kernel.
size_t gemm_pair_small_smem(int m, int k, int n, int p, int nbuf) {
  const SmallGeom g = small_geom(m, k, n, p);
  return sizeof(double) * ((size_t)nbuf * (g.szA + g.szX + g.szB) + g.szT);
}

template <int WPI>
static su2_status launch_small(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, const double* X,
                               const double* B, double* C, int nbuf, int vec_ok, size_t smem, int sms, cudaStream_t stream) {
  cudaError_t e = cudaFuncSetAttribute(gemm_pair_small_kernel<WPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) { set_cuda_error("cudaFuncSetAttribute(gemm_pair_small_kernel)", (int)e); return SU2_ERR_CUDA; }
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gemm_pair_small_kernel<WPI>, 32 * WPI, smem);
  if (e != cudaSuccess || per_sm < 1) { set_cuda_error("occupancy(gemm_pair_small_kernel)", (int)e); return SU2_ERR_CUDA; }
  const int64_t grid = std::min<int64_t>(batch, (int64_t)sms * per_sm);
  gemm_pair_small_kernel<WPI><<<(unsigned)grid, 32 * WPI, smem, stream>>>(m, k, n, p, batch, alpha, A, X, B, C, nbuf, vec_ok);
  e = cudaGetLastError();
  if (e != cudaSuccess) { set_cuda_error("gemm_pair_small_kernel launch", (int)e); return SU2_ERR_CUDA; }
  count_launch();
  return SU2_OK;
}

// Returns SU2_OK after launching, or 1 if the shape does not belong here (caller falls through to the tile
// kernels).  wpi_force / nbuf_force = 0: heuristics below.
su2_status launch_gemm_pair_small(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, const double* X,
                                  const double* B, double* C, void* stream_v, int wpi_force, int nbuf_force) {
  constexpr size_t SMEM_SM = 227 * 1024;
  if (gemm_pair_small_smem(m, k, n, p, 1) > SMEM_SM) return 1;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  // warps per item: 16 x 16 macro tiles of the larger of the two product grids
  const SmallGeom g = small_geom(m, k, n, p);
  const int macro = std::max(((g.M8 + 15) / 16) * ((g.N8 + 15) / 16), ((g.M8 + 15) / 16) * ((g.P8 + 15) / 16));
  // as many warps as there are macro tiles, at most 16 (measured on B200: 48^4 -> 8 warps 13.3 vs 4 warps 10.8
  // TFLOP/s; 64^4 -> 16 warps 17.7 vs 8 warps 14.6; 32^4 -> 4 warps 16.1 vs 8 warps 8.8)
  int wpi = 1;
  while (2 * wpi <= std::min(macro, 16)) wpi *= 2;
  if (macro < 3) wpi = 1;
  if (wpi_force == 1 || wpi_force == 2 || wpi_force == 4 || wpi_force == 8 || wpi_force == 16) wpi = wpi_force;
  // double buffering only while it costs no residency (32 CTAs per SM, +1 KB per CTA reserved by the hardware):
  // measured on B200, occupancy beats prefetch for every shape from 16 x 16 up (b = 16: 6.3 vs 5.4 TB/s)
  int nbuf = (gemm_pair_small_smem(m, k, n, p, 2) + 1024) * 32 <= SMEM_SM ? 2 : 1;
  if (nbuf_force == 1 || nbuf_force == 2) nbuf = nbuf_force;
  const size_t smem = gemm_pair_small_smem(m, k, n, p, nbuf);
  if (smem > SMEM_SM) return 1;
  // 16-byte copies and C updates: even row lengths, 16-byte aligned bases, even item sizes
  const bool even = !(k & 1) && !(n & 1) && !(p & 1);
  const bool aligned = !(((uintptr_t)A | (uintptr_t)X | (uintptr_t)B | (uintptr_t)C) & 15);
  const int vec_ok = even && aligned;
  cudaStream_t stream = (cudaStream_t)stream_v;
  if (wpi == 1) return launch_small<1>(m, k, n, p, batch, alpha, A, X, B, C, nbuf, vec_ok, smem, sms, stream);
  if (wpi == 2) return launch_small<2>(m, k, n, p, batch, alpha, A, X, B, C, nbuf, vec_ok, smem, sms, stream);
  if (wpi == 4) return launch_small<4>(m, k, n, p, batch, alpha, A, X, B, C, nbuf, vec_ok, smem, sms, stream);
  if (wpi == 8) return launch_small<8>(m, k, n, p, batch, alpha, A, X, B, C, nbuf, vec_ok, smem, sms, stream);
  return launch_small<16>(m, k, n, p, batch, alpha, A, X, B, C, nbuf, vec_ok, smem, sms, stream);
}

}  // namespace su2
