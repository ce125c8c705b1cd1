// Strided-batched FP64 GEMM-pair microbenchmark entry (BASELINE.json configs[4]):
//   C_b += alpha * A_b X_b B_b^T, one independent item per batch index.
// Items whose operands fit an SM's shared memory run on the small-block kernel (gemm_pair_small.cu, whole items per
// CTA, many in flight per SM).  Everything else whose rows are 16-byte aligned (even k and n) runs on the fused DMMA
// kernel of the hot path (heff_tma.cu): A, X and B are rank-3 tensors {columns, rows, batch}, three tensor maps
// describe the whole call, a small kernel writes one task / unit / work-item record per batch item (and output
// tile), and the persistent kernel consumes them with the accumulate flag.  Only odd-k / odd-n items too large for
// the small-block kernel fall to the FP64-FMA tile routine below.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "su2_internal.h"
#include "tile_config.h"

namespace su2 {

constexpr int TILE_M = 64;
constexpr int TILE_P = 64;
constexpr int GP_THREADS = 256;
constexpr int NC = 32;    // columns of T (n-chunk) per pass
constexpr int KC = 16;    // k-chunk of the first product

struct TileSmem {
  double As[TILE_M][KC + 1];      // A[row0+i][k0+kk]
  double Es[KC][NC + 1];          // E[k0+kk][n0+j]
  double Ts[TILE_M][NC + 1];      // coef*alpha * (A E)[i][j]
  double Ds[TILE_P][NC + 1];      // D[col0+c][n0+j]
};

// acc (64x64 tile at (row0,col0), thread (ty,tx) owns rows ty+16i, cols tx+16c)
//   += coef * sum_{pos0<=pos<pos1} alpha_pos * A_pos[row0:,:] E D_pos[col0:,:]^T
__device__ __forceinline__ void accumulate_task(const DevTask& t, const double* __restrict__ E, int pos0, int pos1,
                                                int row0, int col0, TileSmem& sm, double (&acc)[4][4]) {
  const int tid = threadIdx.x;
  const int ty = tid / 16, tx = tid % 16;    // second product: rows ty+16*i, cols tx+16*j
  const int gy = tid / 8, gx = tid % 8;      // first product : rows gy+32*i (i<2), cols gx+8*j (j<4)
  const bool ta = t.flags & TASK_TRANS_A, td = t.flags & TASK_TRANS_D;
  for (int pos = pos0; pos < pos1; ++pos) {
    const double* __restrict__ A = t.A + (int64_t)pos * t.strideA;
    const double* __restrict__ D = t.D + (int64_t)pos * t.strideD;
    const double scale = t.coef * (t.alpha ? t.alpha[pos] : 1.0);
    for (int n0 = 0; n0 < t.n; n0 += NC) {
      // ---- first product: T[64 x NC] = A[row0:row0+64, :] * E[:, n0:n0+NC]
      double tacc[2][4];
#pragma unroll
      for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) tacc[i][j] = 0.0;
      for (int k0 = 0; k0 < t.k; k0 += KC) {
        for (int e = tid; e < TILE_M * KC; e += GP_THREADS) {
          int i, kk;
          if (!ta) { i = e / KC; kk = e % KC; } else { kk = e / TILE_M; i = e % TILE_M; }
          const int r = row0 + i, c = k0 + kk;
          double v = 0.0;
          if (r < t.m && c < t.k) v = ta ? A[(int64_t)c * t.ldA + r] : A[(int64_t)r * t.ldA + c];
          sm.As[i][kk] = v;
        }
        for (int e = tid; e < KC * NC; e += GP_THREADS) {
          const int kk = e / NC, j = e % NC;
          const int r = k0 + kk, c = n0 + j;
          sm.Es[kk][j] = (r < t.k && c < t.n) ? E[(int64_t)r * t.n + c] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < KC; ++kk) {
          double a[2], b[4];
#pragma unroll
          for (int i = 0; i < 2; ++i) a[i] = sm.As[gy + 32 * i][kk];
#pragma unroll
          for (int j = 0; j < 4; ++j) b[j] = sm.Es[kk][gx + 8 * j];
#pragma unroll
          for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) tacc[i][j] = fma(a[i], b[j], tacc[i][j]);
        }
        __syncthreads();
      }
#pragma unroll
      for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) sm.Ts[gy + 32 * i][gx + 8 * j] = scale * tacc[i][j];
      // ---- D tile: Ds[c][j] = D[col0+c][n0+j]
      for (int e = tid; e < TILE_P * NC; e += GP_THREADS) {
        int c, j;
        if (!td) { c = e / NC; j = e % NC; } else { j = e / TILE_P; c = e % TILE_P; }
        const int r = col0 + c, q = n0 + j;
        double v = 0.0;
        if (r < t.p && q < t.n) v = td ? D[(int64_t)q * t.ldD + r] : D[(int64_t)r * t.ldD + q];
        sm.Ds[c][j] = v;
      }
      __syncthreads();
      // ---- second product: F_tile += T * Ds^T  (K = NC columns of this position's stripe)
#pragma unroll 8
      for (int j = 0; j < NC; ++j) {
        double a[4], b[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) a[i] = sm.Ts[ty + 16 * i][j];
#pragma unroll
        for (int c = 0; c < 4; ++c) b[c] = sm.Ds[tx + 16 * c][j];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int c = 0; c < 4; ++c) acc[i][c] = fma(a[i], b[c], acc[i][c]);
      }
      __syncthreads();
    }
  }
}

// BASELINE.json configs[4]: C_b += alpha A_b X_b B_b^T; blockIdx.x = tile, blockIdx.y/z = batch index.
__global__ void __launch_bounds__(GP_THREADS)
gemm_pair_kernel(int m, int k, int n, int p, int64_t batch, double alpha, const double* __restrict__ A,
                 const double* __restrict__ X, const double* __restrict__ B, double* __restrict__ C) {
  __shared__ TileSmem sm;
  const int tiles_p = (p + TILE_P - 1) / TILE_P;
  const int row0 = (blockIdx.x / tiles_p) * TILE_M, col0 = (blockIdx.x % tiles_p) * TILE_P;
  const int ty = threadIdx.x / 16, tx = threadIdx.x % 16;
  for (int64_t b = blockIdx.y; b < batch; b += gridDim.y) {
    DevTask t;
    t.A = A + b * (int64_t)m * k; t.D = B + b * (int64_t)p * n; t.alpha = nullptr; t.coef = alpha; t.e_off = 0;
    t.m = m; t.k = k; t.n = n; t.p = p; t.strideA = 0; t.strideD = 0; t.ldA = k; t.ldD = n; t.npos = 1; t.flags = 0;
    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
    accumulate_task(t, X + b * (int64_t)k * n, 0, 1, row0, col0, sm, acc);
    double* __restrict__ dst = C + b * (int64_t)m * p;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const int r = row0 + ty + 16 * i, q = col0 + tx + 16 * c;
        if (r < m && q < p) dst[(int64_t)r * p + q] += acc[i][c];
      }
  }
}


// rows of `cols` doubles (pitch cols) -> rows of pitch ld (> cols); the pad columns are never read (the tensor maps keep the
// true extent, out-of-bounds columns are zero-filled by the copy engine)
__global__ void __launch_bounds__(256) repitch_kernel(const double* __restrict__ src, double* __restrict__ dst, int64_t rows, int cols, int ld) {
  // one warp per row (no division per element), lanes along the row
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t r = warp0; r < rows; r += nwarp) {
    const double* __restrict__ s = src + r * cols;
    double* __restrict__ d = dst + r * ld;
    for (int c = lane; c < cols; c += 32) d[c] = s[c];
  }
}

// one task, one unit and ntile work items per batch index; the batch index is the item coordinate of the three
// tensor maps (A, X, B are rank-3 tensors {columns, rows, batch})
__global__ void gemm_pair_tables_kernel(int m, int k, int n, int p, int64_t batch, double alpha, int wr, int tm, int tp,
                                        DevTask* tasks, DevUnit* units, DevWork* work, int* counter) {
  const int tr = (m + tm - 1) / tm, tc = (p + tp - 1) / tp;
  if (blockIdx.x == 0 && threadIdx.x == 0) *counter = 0;
  for (int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; b < batch; b += (int64_t)gridDim.x * blockDim.x) {
    DevTask t;
    t.A = nullptr; t.D = nullptr; t.alpha = nullptr; t.coef = alpha;
    t.e_off = b * (int64_t)k * n; t.m = m; t.k = k; t.n = n; t.p = p;
    t.strideA = m * k; t.strideD = p * n; t.ldA = k; t.ldD = n; t.npos = 1; t.flags = 0;
    t.mapA = 0; t.mapD = 1; t.mapE = 2; t.e_item = (int32_t)b; t.ldE = n; t.pad = 0;
    tasks[b] = t;
    units[b] = DevUnit{(int32_t)b, (int32_t)b, (int32_t)b + 1, 0};     // "position" b = the item coordinate of A and B
    for (int i = 0; i < tr * tc; ++i) {
      DevWork w;
      w.dst_off = b * (int64_t)m * p; w.unit0 = (int32_t)b; w.unit1 = (int32_t)b + 1;
      w.row0 = (i / tc) * tm; w.col0 = (i % tc) * tp; w.m = m; w.p = p; w.to_partial = 2; w.wr = wr; w.ldo = p; w.gang = -1;
      work[b * (int64_t)(tr * tc) + i] = w;
    }
  }
}

su2_status launch_gemm_pair(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, const double* X,
                            const double* B, double* C, void* stream_v, int route, int wpi, int nbuf) {
  if (batch == 0) return SU2_OK;
  cudaStream_t stream = (cudaStream_t)stream_v;
  // automatic choice: items of at least 48 in every extent run un-fused on the two-pass GEMM (gemm_two_pass.cu) -- measured on
  // one B200, TFLOP/s un-fused / best other route: 48^4 16.5 / 13.4, 64^4 21.1 / 17.7, 96^4 25.8 / 12.6, 128^4 27.1 / 19.1,
  // 192^4 29.6 / 21.1, 256^4 30.5 / 22.5, 512^4 32.7 / 26.2, 547^4 27.5 / 23.7 (odd row lengths re-pitched inside); 32^4
  // 9.1 / 16.2 stays on the small-block kernel, and so do items with one short extent (8 x 512 x 512 x 8)
  constexpr int TWO_PASS_MIN_EXTENT = 48;
  if (route == 0 && std::min(std::min(m, k), std::min(n, p)) >= TWO_PASS_MIN_EXTENT) route = 4;
  if (route == 0 || route == 1) {
    // items whose operands fit one SM's shared memory (all dims <= 80 for square shapes): one CTA of 1-16 warps per
    // item, shared memory sized by the item shape (gemm_pair_small.cu)
    su2_status st = launch_gemm_pair_small(m, k, n, p, batch, alpha, A, X, B, C, stream_v, wpi, nbuf);
    if (st != 1) return st;
    if (route == 1) return SU2_ERR_INVALID_ARGUMENT;
  }
  // anything else whose rows are 16-byte aligned runs on the fused kernel of the apply (heff_tma.cu): the three
  // operands are rank-3 tensors {columns, rows, batch}, so three tensor maps describe the whole call
  // Bulk-tensor copies need 16-byte aligned rows.  An operand with an odd row length (or an odd base address) is copied once
  // into a stream-ordered buffer with an even row pitch -- 16 bytes of traffic per element against 2 x (row length) flops --
  // instead of sending the whole call to the FP64-FMA routine (1.4 TFLOP/s at 547^4 against 25 on this route).
  const bool padA = (k & 1) || ((uintptr_t)A & 15), padX = (n & 1) || ((uintptr_t)X & 15), padB = (n & 1) || ((uintptr_t)B & 15);
  const int ldA = k + (k & 1), ldX = n + (n & 1), ldB = n + (n & 1);
  const int64_t max_items = (int64_t)1 << 24;
  // (the automatic choice of route 4 is made at the top: every extent >= TWO_PASS_MIN_EXTENT)
  if (route == 4) {
    // un-fused form (gemm_two_pass.cu): T through a scratch, both passes with 32 x 64 warp tiles and two CTAs per SM
    const size_t b_padA = padA ? (((size_t)batch * m * ldA * 8 + 255) & ~(size_t)255) : 0;
    const size_t b_padX = padX ? (((size_t)batch * k * ldX * 8 + 255) & ~(size_t)255) : 0;
    const size_t b_padB = padB ? (((size_t)batch * p * ldB * 8 + 255) & ~(size_t)255) : 0;
    char* pads = nullptr;
    if (b_padA + b_padX + b_padB) {
      su2_status sp = gemm_scratch_alloc((void**)&pads, b_padA + b_padX + b_padB, stream_v);   // the pool of gemm_two_pass.cu
      if (sp != SU2_OK) return sp;
    }
    const double *mA = A, *mX = X, *mB = B;
    auto repitch = [&](const double* src, char* dst, int64_t rows, int cols, int ld) {
      repitch_kernel<<<(unsigned)std::min<int64_t>((rows + 7) / 8, 148 * 32), 256, 0, stream>>>(src, (double*)dst, rows, cols, ld);
      count_launch();
      return (const double*)dst;
    };
    if (padA) mA = repitch(A, pads, (int64_t)batch * m, k, ldA);
    if (padX) mX = repitch(X, pads + b_padA, (int64_t)batch * k, n, ldX);
    if (padB) mB = repitch(B, pads + b_padA + b_padX, (int64_t)batch * p, n, ldB);
    su2_status st = launch_gemm_two_pass(m, k, n, p, batch, alpha, mA, padA ? ldA : k, mX, padX ? ldX : n, mB, padB ? ldB : n, C, stream_v);
    if (pads) cudaFreeAsync(pads, stream);
    return st;
  }
  if ((route == 0 || route == 2) && batch < max_items) {
    // tile class with the lowest modelled cost, like the planner
    int wr = 1;
    double best = -1.0;
    for (int cand : {1, 2, 4}) {
      const TileShape ts = tile_shape(cand);
      double c = 0.0;
      for (int r0 = 0; r0 < m; r0 += ts.tm)
        for (int c0 = 0; c0 < p; c0 += ts.tp) c += tile_pos_cost(cand, std::min(ts.tm, m - r0), std::min(ts.tp, p - c0), k, n);
      if (best < 0.0 || c < best) { best = c; wr = cand; }
    }
    const TileShape ts = tile_shape(wr);
    const int64_t ntile = (int64_t)((m + ts.tm - 1) / ts.tm) * ((p + ts.tp - 1) / ts.tp);
    if (batch * ntile < ((int64_t)1 << 31)) {
      alignas(128) unsigned char h_maps[3 * 128];
      const int nb = (int)batch;
      su2_status st;
      const size_t b_maps = 512;
      const size_t b_task = ((size_t)batch * sizeof(DevTask) + 255) & ~(size_t)255;
      const size_t b_unit = ((size_t)batch * sizeof(DevUnit) + 255) & ~(size_t)255;
      const size_t b_work = ((size_t)(batch * ntile) * sizeof(DevWork) + 255) & ~(size_t)255;
      const size_t b_padA = padA ? (((size_t)batch * m * ldA * 8 + 255) & ~(size_t)255) : 0;
      const size_t b_padX = padX ? (((size_t)batch * k * ldX * 8 + 255) & ~(size_t)255) : 0;
      const size_t b_padB = padB ? (((size_t)batch * p * ldB * 8 + 255) & ~(size_t)255) : 0;
      char* buf = nullptr;
      cudaError_t e = cudaMallocAsync((void**)&buf, b_maps + b_task + b_unit + b_work + 256 + b_padA + b_padX + b_padB, stream);
      if (e != cudaSuccess) { set_cuda_error("cudaMallocAsync(gemm_pair tables)", (int)e); return SU2_ERR_CUDA; }
      char* pads = buf + b_maps + b_task + b_unit + b_work + 256;
      const double *mA = A, *mX = X, *mB = B;
      auto repitch = [&](const double* src, char* dst, int64_t rows, int cols, int ld) {
        repitch_kernel<<<(unsigned)std::min<int64_t>((rows + 7) / 8, 148 * 32), 256, 0, stream>>>(src, (double*)dst, rows, cols, ld);
        count_launch();
        return (const double*)dst;
      };
      if (padA) mA = repitch(A, pads, (int64_t)batch * m, k, ldA);
      if (padX) mX = repitch(X, pads + b_padA, (int64_t)batch * k, n, ldX);
      if (padB) mB = repitch(B, pads + b_padA + b_padX, (int64_t)batch * p, n, ldB);
      e = cudaGetLastError();
      if (e != cudaSuccess) { set_cuda_error("repitch_kernel launch", (int)e); cudaFreeAsync(buf, stream); return SU2_ERR_CUDA; }
      if ((st = encode_tensor_map(h_maps, MapKey{mA, m, k, padA ? ldA : k, nb, (int64_t)m * (padA ? ldA : k), KS1, ts.tm})) != SU2_OK ||
          (st = encode_tensor_map(h_maps + 128, MapKey{mB, p, n, padB ? ldB : n, nb, (int64_t)p * (padB ? ldB : n), KS2, DBOX_C})) != SU2_OK ||
          (st = encode_tensor_map(h_maps + 256, MapKey{mX, k, n, padX ? ldX : n, nb, (int64_t)k * (padX ? ldX : n), EBOX_LD, KS1})) != SU2_OK) {
        cudaFreeAsync(buf, stream);
        return st;
      }
      DevTask* tasks = (DevTask*)(buf + b_maps);
      DevUnit* units = (DevUnit*)(buf + b_maps + b_task);
      DevWork* work = (DevWork*)(buf + b_maps + b_task + b_unit);
      int* counter = (int*)(buf + b_maps + b_task + b_unit + b_work);
      // pageable source: the runtime stages the 384 bytes before the call returns
      e = cudaMemcpyAsync(buf, h_maps, sizeof(h_maps), cudaMemcpyHostToDevice, stream);
      if (e != cudaSuccess) { set_cuda_error("cudaMemcpyAsync(gemm_pair tensor maps)", (int)e); cudaFreeAsync(buf, stream); return SU2_ERR_CUDA; }
      gemm_pair_tables_kernel<<<(unsigned)std::min<int64_t>((batch + 127) / 128, 1024), 128, 0, stream>>>(
          m, k, n, p, batch, alpha, wr, ts.tm, ts.tp, tasks, units, work, counter);
      e = cudaGetLastError();
      if (e != cudaSuccess) { set_cuda_error("gemm_pair_tables_kernel launch", (int)e); cudaFreeAsync(buf, stream); return SU2_ERR_CUDA; }
      count_launch();
      int dev = 0, sms = 148;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
      st = launch_heff_tma_tables(work, (int)(batch * ntile), units, tasks, buf, C, nullptr, counter, nullptr, sms, stream_v);
      cudaFreeAsync(buf, stream);
      return st;
    }
  }
  if (route == 2) return SU2_ERR_INVALID_ARGUMENT;
  // rows that are not 16-byte aligned (odd k or n) and too large for the small-block kernel: FP64-FMA tile routine
  const int tiles = ((m + TILE_M - 1) / TILE_M) * ((p + TILE_P - 1) / TILE_P);
  dim3 grid(tiles, (unsigned)std::min<int64_t>(batch, 65535));
  gemm_pair_kernel<<<grid, GP_THREADS, 0, stream>>>(m, k, n, p, batch, alpha, A, X, B, C);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_cuda_error("gemm_pair_kernel launch", (int)e); return SU2_ERR_CUDA; }
  count_launch();
  return SU2_OK;
}

}  // namespace su2

extern "C" su2_status su2_gemm_pair_batched(int32_t m, int32_t k, int32_t n, int32_t p, int64_t batch, double alpha,
                                            const double* A, const double* X, const double* B, double* C,
                                            void* cuda_stream) {
  if (m <= 0 || k <= 0 || n <= 0 || p <= 0 || batch < 0 || !A || !X || !B || !C) return SU2_ERR_INVALID_ARGUMENT;
  return su2::launch_gemm_pair(m, k, n, p, batch, alpha, A, X, B, C, cuda_stream, 0, 0, 0);
}

extern "C" su2_status su2_gemm_pair_batched_route(int32_t m, int32_t k, int32_t n, int32_t p, int64_t batch, double alpha,
                                                  const double* A, const double* X, const double* B, double* C,
                                                  void* cuda_stream, int32_t route, int32_t wpi, int32_t nbuf) {
  if (m <= 0 || k <= 0 || n <= 0 || p <= 0 || batch < 0 || !A || !X || !B || !C || route < 0 || route > 4)
    return SU2_ERR_INVALID_ARGUMENT;
  return su2::launch_gemm_pair(m, k, n, p, batch, alpha, A, X, B, C, cuda_stream, route, wpi, nbuf);
}
