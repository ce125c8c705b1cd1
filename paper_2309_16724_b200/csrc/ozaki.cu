// libsu2ozaki.so (include/su2_ozaki.h): the strided-batched FP64 GEMM pair on the INT8 tensor path
// (the FP64 ceiling the paper's headline is quoted against).
//
// tcgen05.mma has no f64 kind and DMMA runs at the DFMA rate on sm_100a (37 TFLOP/s), so the road past that ceiling with
// tensor units is exact integer arithmetic on tcgen05.mma kind::i8 (int32 accumulators in TMEM).  Per product L (M x K) . R (K x N),
// following oracle/ozaki.py step by step:
//   1. every row of L and every column of R is scaled by a power of two to |v| < 1 (exponents e_i, f_j);
//   2. and cut into S slices of 7 bits by truncation (INT8 in [-127, 127]);
//   3. the slice pairs (s, t) with s + t = d are ONE exact INT8 GEMM with int32 accumulation over the concatenated
//      contraction index of length (d+1) K: L's slices are stored 0..S-1 along its rows, R's slices S-1..0 along its
//      contraction index, so a diagonal is a prefix window of one and a suffix window of the other -- S GEMMs, S(S+1)/2 pairs;
//   4. the S integer planes are recombined in FP64, smallest first, and scaled by 2^(e_i + f_j).
// The pair C += alpha (A X) B^T runs product 1 with R = X as stored (rows = contraction index: an MN-major INT8 operand, no
// transposition) and product 2 with R = B^T (B's rows are K-major as stored).  Recombining product 1 and slicing its result T for
// product 2 is one kernel (T is never written in FP64).
//
// The INT8 GEMM is generated from the CUTLASS 4.x sm_100 collective builder (vendored CuTe/CUTLASS header templates: TMA loads,
// tcgen05.mma.cta_group::{1,2}.kind::i8 issued by one thread, TMEM accumulators, SASS UTCIMMA); everything else here is hand-written.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstring>

#include "cutlass/cutlass.h"
#include "cute/tensor.hpp"
#include "cutlass/gemm/device/gemm_universal_adapter.h"
#include "cutlass/gemm/kernel/gemm_universal.hpp"
#include "cutlass/gemm/collective/collective_builder.hpp"
#include "cutlass/epilogue/collective/collective_builder.hpp"

#include "su2_ozaki.h"

namespace su2oz {

constexpr int OZ_W = 7;                     // bits per slice
constexpr int OZ_SMAX = SU2_OZAKI_MAX_SLICES;
constexpr int OZ_OK = 0, OZ_INVALID = -1, OZ_CUDA = -5;

thread_local char g_err[256] = "";
std::atomic<int64_t> g_launches{0};

int fail(int code, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
  else snprintf(g_err, sizeof(g_err), "%s", what);
  return code;
}

// v 2^e, exact (ldexp); the factor 2^e is built from its bits when it is a normal number, which gives ldexp's result in one
// multiplication (a power-of-two factor is exact, and where the product is subnormal both round the same way)
__device__ __forceinline__ double scale2(double v, int e) {
  return (e >= -1022 && e <= 1023) ? v * __hiloint2double((1023 + e) << 20, 0) : ldexp(v, e);
}

// |a| as an ordered integer: for finite doubles the order of the bit patterns of |a| is the order of the magnitudes
__device__ __forceinline__ unsigned long long abs_bits(double a) { return (unsigned long long)__double_as_longlong(a) & 0x7fffffffffffffffull; }

// exponent of the scaling of a line whose largest magnitude has the bit pattern amax: amax 2^-e in [0.5, 1); 0 for a zero line
// (oracle/ozaki.py step 1: floor(log2 amax) + 1).  Normal numbers read it off the exponent field.
__device__ __forceinline__ int line_exponent(unsigned long long amax) {
  if (amax == 0) return 0;
  const int E = (int)(amax >> 52);
  if (E) return E - 1022;
  int e;
  (void)frexp(__longlong_as_double((long long)amax), &e);      // subnormal maximum
  return e;
}

// The S slices of v = a 2^-e (|v| < 1) by truncation toward zero (oracle/ozaki.py step 2: t = 128 v; q = trunc(t); t -= q; ...).
// Every step of that recurrence is exact, so the slices are the base-128 digits of |v|, signed: with a = +-M 2^(E-1075)
// (M the 53-bit significand), floor(|v| 2^(7S)) = M >> (1075 - 7S + e - E) and q_s = +-((that >> 7(S-1-s)) & 127) -- integer
// shifts instead of 4 S dependent FP64 operations per element (the slicing kernels were bound by the FP64 pipe).
template <int S>
__device__ __forceinline__ void slices_of(double a, int e, int8_t (&q)[OZ_SMAX]) {
  const long long bits = __double_as_longlong(a);
  int E = (int)((bits >> 52) & 0x7ff);
  unsigned long long M = (unsigned long long)bits & 0xfffffffffffffull;
  if (E) M |= 1ull << 52; else E = 1;                           // subnormal: no hidden bit, exponent of the smallest normal
  const int sh = 1075 - OZ_W * S + e - E;                       // >= 53 - 7 S > 0 because |v| < 1
  const unsigned long long fx = sh < 64 ? M >> sh : 0ull;
  const int sgn = bits < 0 ? -1 : 1;
#pragma unroll
  for (int s = 0; s < S; ++s) q[s] = (int8_t)(sgn * (int)((fx >> (OZ_W * (S - 1 - s))) & 127));
}

// 4 consecutive elements of a line from element j on, zeros from `len` on; vec: the line starts on a 16-byte boundary
__device__ __forceinline__ void load4(const double* __restrict__ row, int j, int len, bool vec, double (&v)[4]) {
  if (vec && j + 3 < len) {
    const double2 a = *(const double2*)(row + j), b = *(const double2*)(row + j + 2);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
  } else {
#pragma unroll
    for (int q = 0; q < 4; ++q) v[q] = (j + q < len) ? row[j + q] : 0.0;
  }
}

__device__ __forceinline__ unsigned long long amax4(unsigned long long a, const double (&v)[4]) {
  return max(max(a, max(abs_bits(v[0]), abs_bits(v[1]))), max(abs_bits(v[2]), abs_bits(v[3])));
}

// Shapes need not be multiples of anything: the INT8 copies are this file's own, so their extents are padded (contraction
// lengths and MN-major rows to 16 bytes for TMA, int32 plane rows to 16 bytes) and the pads are written as zeros, which add
// nothing to the integer sums.  FP64 operands are read with 16-byte loads where a line is aligned, element-wise otherwise.

// ---- slicing of a K-major operand: one warp per line ------------------------------------------------------------------------------
// src: items of `rows` lines of `len` FP64 (line pitch ld, items istride apart).  The INT8 copy has rowsP >= rows lines per item
// (lines beyond `rows` are zero: B's rows are padded to a multiple of 4) of S slots of lenP >= len bytes: slice s of element j
// of line r of item b goes to q[((b rowsP + r) S + slot(s)) lenP + j], slot(s) = s (left operand) or S-1-s (REVERSED: right
// operand); expo[b rowsP + r] = the line's exponent.  Each lane owns 4 consecutive elements (one 4-byte store per slice).
template <int S, bool REVERSED>
__global__ void __launch_bounds__(256)
slice_rows_kernel(const double* __restrict__ src, int64_t istride, int64_t ld, int rows, int rowsP, int len, int lenP, int64_t nlines,
                  int8_t* __restrict__ q, int32_t* __restrict__ expo) {
  const int lane = threadIdx.x & 31;
  const int64_t line = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (line >= nlines) return;
  const int64_t item = line / rowsP;
  const int r = (int)(line - item * rowsP);
  int8_t* __restrict__ out = q + line * (int64_t)S * lenP;
  if (r >= rows) {                                            // padding line
    if (lane == 0) expo[line] = 0;
    for (int j = lane * 4; j < S * lenP; j += 128) *(char4*)(out + j) = make_char4(0, 0, 0, 0);
    return;
  }
  const double* __restrict__ row = src + item * istride + (int64_t)r * ld;
  const bool vec = ((uintptr_t)row & 15) == 0;
  unsigned long long amax = 0;
  for (int j = lane * 4; j < len; j += 128) {
    double v[4];
    load4(row, j, len, vec, v);
    amax = amax4(amax, v);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) amax = max(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  const int e = line_exponent(amax);
  if (lane == 0) expo[line] = e;
  for (int j = lane * 4; j < lenP; j += 128) {
    double v[4];
    load4(row, j, len, vec, v);
    int8_t q0[OZ_SMAX], q1[OZ_SMAX], q2[OZ_SMAX], q3[OZ_SMAX];
    slices_of<S>(v[0], e, q0); slices_of<S>(v[1], e, q1); slices_of<S>(v[2], e, q2); slices_of<S>(v[3], e, q3);
#pragma unroll
    for (int s = 0; s < S; ++s)
      *(char4*)(out + (int64_t)(REVERSED ? S - 1 - s : s) * lenP + j) = make_char4(q0[s], q1[s], q2[s], q3[s]);
  }
}

// ---- slicing of an MN-major operand (the contraction index runs down the rows of the stored block): one CTA per (128-column strip, item)
// src: items (istride apart) of k rows of n FP64, row pitch ld.  expo[item nP + c] = exponent of column c (0 for the padding
// columns); slice s of element (j, c) goes to q[item][slot(s) kP + j][c] (row pitch nP), slot(s) = S-1-s for a right operand
// (REVERSED: X as stored, D stored transposed) or s for a left operand (A stored transposed: an M-major left operand); rows
// k..kP-1 and columns n..nP-1 are zero.
template <int S, bool REVERSED>
__global__ void __launch_bounds__(256)
slice_cols_kernel(const double* __restrict__ src, int64_t istride, int64_t ld, int k, int n, int kP, int nP, int8_t* __restrict__ q,
                  int32_t* __restrict__ expo) {
  __shared__ unsigned long long s_amax[8][128];
  __shared__ int s_e[128];
  const int lane = threadIdx.x & 31, wy = threadIdx.x >> 5;
  const int64_t item = blockIdx.y;
  const int c = blockIdx.x * 128 + lane * 4;
  const bool live = c < nP;                                  // nP % 4 == 0: a thread's 4 columns are all inside or all outside
  const double* __restrict__ x = src + item * istride;
  const bool vec = !(ld & 1) && ((uintptr_t)x & 15) == 0;    // every row of this item starts on a 16-byte boundary
  unsigned long long a[4] = {0, 0, 0, 0};
  if (live)
    for (int j = wy; j < k; j += 8) {
      double v[4];
      load4(x + (int64_t)j * ld, c, n, vec, v);
#pragma unroll
      for (int u = 0; u < 4; ++u) a[u] = max(a[u], abs_bits(v[u]));
    }
#pragma unroll
  for (int u = 0; u < 4; ++u) s_amax[wy][lane * 4 + u] = a[u];
  __syncthreads();
  if (threadIdx.x < 128) {
    unsigned long long m = 0;
#pragma unroll
    for (int y = 0; y < 8; ++y) m = max(m, s_amax[y][threadIdx.x]);
    const int e = line_exponent(m);
    s_e[threadIdx.x] = e;
    if (blockIdx.x * 128 + threadIdx.x < nP) expo[item * nP + blockIdx.x * 128 + threadIdx.x] = e;
  }
  __syncthreads();
  if (!live) return;
  const int e0 = s_e[lane * 4], e1 = s_e[lane * 4 + 1], e2 = s_e[lane * 4 + 2], e3 = s_e[lane * 4 + 3];
  int8_t* __restrict__ out = q + item * (int64_t)S * kP * nP;
  for (int j = wy; j < kP; j += 8) {
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    if (j < k) load4(x + (int64_t)j * ld, c, n, vec, v);
    int8_t q0[OZ_SMAX], q1[OZ_SMAX], q2[OZ_SMAX], q3[OZ_SMAX];
    slices_of<S>(v[0], e0, q0); slices_of<S>(v[1], e1, q1); slices_of<S>(v[2], e2, q2); slices_of<S>(v[3], e3, q3);
#pragma unroll
    for (int s = 0; s < S; ++s)
      *(char4*)(out + ((int64_t)(REVERSED ? S - 1 - s : s) * kP + j) * nP + c) = make_char4(q0[s], q1[s], q2[s], q3[s]);
  }
}

// ---- recombination -----------------------------------------------------------------------------------------------------------------
// value of 4 consecutive entries of the product from their S integer planes (plane d at planes + d * plane_stride), before the
// 2^(e+f) scaling:  sum_{d = S-1 .. 0} P_d 2^(-W (d+2)),  smallest first (oracle/ozaki.py step 5); the weights are powers of two, so
// multiplying is exact.  idx is a multiple of 4 (plane rows are padded to 4 entries).
template <int S>
__device__ __forceinline__ void combine4(const int32_t* __restrict__ planes, int64_t plane_stride, int64_t idx, double (&v)[4]) {
  v[0] = v[1] = v[2] = v[3] = 0.0;
#pragma unroll
  for (int d = S - 1; d >= 0; --d) {
    const int4 pl = *(const int4*)(planes + d * plane_stride + idx);
    const double w = __hiloint2double((1023 - OZ_W * (d + 2)) << 20, 0);
    v[0] += (double)pl.x * w; v[1] += (double)pl.y * w; v[2] += (double)pl.z * w; v[3] += (double)pl.w * w;
  }
}

// product 1's planes -> slices of T for product 2 (left operand), one warp per row of T.  Plane rows, the column exponents and
// the INT8 rows all have the padded pitch nP; the padding columns hold zero planes and zero exponents, so they come out as zero
// slices without a special case.  T_ij = 2^(e_i + f_j) sum_d ...; row exponent g_i from max_j |T_ij|; slices of T_ij 2^(-g_i) at
// qT[(row S + s) nP + j].  T is never stored in FP64: rows of up to 128 NSTEP columns stay in registers between the exponent
// pass and the slicing pass (NSTEP = 1, 2, 4, 8); longer rows (NSTEP = 0) are recombined twice, the second read of the planes
// coming from L1/L2 (64 FP64 registers per lane for 2048 columns measured slower than the second read).
template <int S, int NSTEP>
__global__ void __launch_bounds__(256)
combine_slice_kernel(const int32_t* __restrict__ planes, int64_t plane_stride, int rows, int nP, int64_t nlines,
                     const int32_t* __restrict__ e_row, int e_pitch, const int32_t* __restrict__ f_col, int f_pitch,
                     int8_t* __restrict__ qT, int32_t* __restrict__ g_row) {
  const int lane = threadIdx.x & 31;
  const int64_t line = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (line >= nlines) return;
  const int64_t item = line / rows;
  const int e = e_row[item * e_pitch + (line - item * rows)];      // pitch 0: one operand shared by all items
  const int32_t* __restrict__ f = f_col + item * f_pitch;
  int8_t* __restrict__ out = qT + line * (int64_t)S * nP;
  // T_ij for the 4 columns at j, exactly as the oracle forms it: the recombined sum, then one scaling by 2^(e_i + f_j)
  auto t_at = [&](int j, double (&t)[4]) {
    combine4<S>(planes, plane_stride, line * nP + j, t);
    const int4 fj = *(const int4*)(f + j);
    t[0] = scale2(t[0], e + fj.x); t[1] = scale2(t[1], e + fj.y); t[2] = scale2(t[2], e + fj.z); t[3] = scale2(t[3], e + fj.w);
  };
  auto put = [&](int j, const double (&t)[4], int g) {
    int8_t q0[OZ_SMAX], q1[OZ_SMAX], q2[OZ_SMAX], q3[OZ_SMAX];
    slices_of<S>(t[0], g, q0); slices_of<S>(t[1], g, q1); slices_of<S>(t[2], g, q2); slices_of<S>(t[3], g, q3);
#pragma unroll
    for (int s = 0; s < S; ++s) *(char4*)(out + (int64_t)s * nP + j) = make_char4(q0[s], q1[s], q2[s], q3[s]);
  };
  unsigned long long amax = 0;
  if constexpr (NSTEP > 0) {
    double t[NSTEP][4];
#pragma unroll
    for (int u = 0; u < NSTEP; ++u) {
      const int j = lane * 4 + u * 128;
      if (j < nP) {
        t_at(j, t[u]);
        amax = amax4(amax, t[u]);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = max(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    const int g = line_exponent(amax);
    if (lane == 0) g_row[line] = g;
#pragma unroll
    for (int u = 0; u < NSTEP; ++u) {
      const int j = lane * 4 + u * 128;
      if (j < nP) put(j, t[u], g);
    }
  } else {
    for (int j = lane * 4; j < nP; j += 128) {
      double t[4];
      t_at(j, t);
      amax = amax4(amax, t);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = max(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    const int g = line_exponent(amax);
    if (lane == 0) g_row[line] = g;
    for (int j = lane * 4; j < nP; j += 128) {
      double t[4];
      t_at(j, t);
      put(j, t, g);
    }
  }
}

// planes of a product -> FP64 result: dst = (ACCUMULATE ? dst : 0) + alpha 2^(e_i + f_j) sum_d ...; 4 consecutive columns per
// thread.  Plane rows and column exponents have the padded pitch colsP; dst is dense (pitch cols).
template <int S, bool ACCUMULATE>
__global__ void __launch_bounds__(256)
combine_out_kernel(const int32_t* __restrict__ planes, int64_t plane_stride, int rows, int cols, int colsP, int64_t nquad,
                   const int32_t* __restrict__ e_row, const int32_t* __restrict__ f_col, double alpha, double* __restrict__ dst) {
  const int cq = colsP >> 2;
  const bool vec = !(cols & 3) && ((uintptr_t)dst & 15) == 0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nquad; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t line = t / cq;                              // item * rows + i
    const int j = (int)(t - line * cq) * 4;
    if (j >= cols) continue;
    const int64_t item = line / rows;
    double v[4];
    combine4<S>(planes, plane_stride, line * colsP + j, v);
    const int e = e_row[line];
    const int4 fj = *(const int4*)(f_col + item * colsP + j);
    v[0] = alpha * scale2(v[0], e + fj.x); v[1] = alpha * scale2(v[1], e + fj.y);
    v[2] = alpha * scale2(v[2], e + fj.z); v[3] = alpha * scale2(v[3], e + fj.w);
    double* o = dst + line * cols + j;
    if (vec) {
      double2 lo = ACCUMULATE ? ((double2*)o)[0] : make_double2(0.0, 0.0), hi = ACCUMULATE ? ((double2*)o)[1] : make_double2(0.0, 0.0);
      lo.x += v[0]; lo.y += v[1]; hi.x += v[2]; hi.y += v[3];
      ((double2*)o)[0] = lo; ((double2*)o)[1] = hi;
    } else {
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (j + u < cols) o[u] = ACCUMULATE ? o[u] + v[u] : v[u];
    }
  }
}

// ---- the exact INT8 GEMM: D (M x N, int32, row-major) = L . R, batched.  L is M x K with K contiguous (LMajorM = false: slices of
// rows) or K x M with M contiguous (true: slices of an operand stored transposed); R is K x N with N contiguous (RMajorN = true:
// X as stored) or N x K with K contiguous (false: B as stored).  Two tile configurations: 256 x 256 x 128 on a pair of SMs
// (cta_group::2, cluster 2 x 1) for outputs of at least 256 x 256, 128 x 128 x 128 on one SM below that.
template <int TM, int TN, int CM>
struct I8Config {
  using Tile = cute::Shape<cute::Int<TM>, cute::Int<TN>, cute::_128>;
  using Cluster = cute::Shape<cute::Int<CM>, cute::_1, cute::_1>;
  using Epilogue = typename cutlass::epilogue::collective::CollectiveBuilder<
      cutlass::arch::Sm100, cutlass::arch::OpClassTensorOp, Tile, Cluster, cutlass::epilogue::collective::EpilogueTileAuto, int32_t,
      int32_t, int32_t, cutlass::layout::RowMajor, 4, int32_t, cutlass::layout::RowMajor, 4,
      cutlass::epilogue::collective::EpilogueScheduleAuto>::CollectiveOp;
  template <class LayoutL, class LayoutR>
  using Mainloop = typename cutlass::gemm::collective::CollectiveBuilder<
      cutlass::arch::Sm100, cutlass::arch::OpClassTensorOp, int8_t, LayoutL, 16, int8_t, LayoutR, 16, int32_t, Tile,
      Cluster, cutlass::gemm::collective::StageCountAutoCarveout<static_cast<int>(sizeof(typename Epilogue::SharedStorage))>,
      cutlass::gemm::collective::KernelScheduleAuto>::CollectiveOp;
  template <class LayoutL, class LayoutR>
  using Gemm = cutlass::gemm::device::GemmUniversalAdapter<
      cutlass::gemm::kernel::GemmUniversal<cute::Shape<int, int, int, int>, Mainloop<LayoutL, LayoutR>, Epilogue>>;
};
using I8Small = I8Config<128, 128, 1>;
using I8Large = I8Config<256, 256, 2>;

template <class Cfg, bool LMajorM, bool RMajorN>
int i8_gemm_cfg(int M, int N, int K, int L, const int8_t* Lp, int64_t ldl, int64_t batchL, const int8_t* Rp, int64_t ldr, int64_t batchR,
                int32_t* D, int64_t batchD, cudaStream_t stream) {
  using Gemm = typename Cfg::template Gemm<std::conditional_t<LMajorM, cutlass::layout::ColumnMajor, cutlass::layout::RowMajor>,
                                           std::conditional_t<RMajorN, cutlass::layout::RowMajor, cutlass::layout::ColumnMajor>>;
  typename Gemm::GemmKernel::StrideA sa;
  if constexpr (LMajorM) sa = cute::make_stride(cute::Int<1>{}, ldl, batchL);       // (M, K, L): M contiguous
  else sa = cute::make_stride(ldl, cute::Int<1>{}, batchL);                          // (M, K, L): K contiguous
  typename Gemm::GemmKernel::StrideB sb;
  if constexpr (RMajorN) sb = cute::make_stride(cute::Int<1>{}, ldr, batchR);       // (N, K, L): N contiguous
  else sb = cute::make_stride(ldr, cute::Int<1>{}, batchR);                          // (N, K, L): K contiguous
  typename Gemm::GemmKernel::StrideD sd = cute::make_stride((int64_t)N, cute::Int<1>{}, batchD);
  typename Gemm::Arguments args{cutlass::gemm::GemmUniversalMode::kGemm, {M, N, K, L}, {Lp, sa, Rp, sb}, {{1, 0}, D, sd, D, sd}};
  Gemm gemm;
  if (gemm.can_implement(args) != cutlass::Status::kSuccess) return fail(OZ_INVALID, "INT8 GEMM: extents or alignment not supported");
  if (Gemm::get_workspace_size(args) != 0) return fail(OZ_CUDA, "INT8 GEMM: unexpected workspace request");
  if (gemm.initialize(args, nullptr, stream) != cutlass::Status::kSuccess) return fail(OZ_CUDA, "INT8 GEMM: initialize", cudaGetLastError());
  if (gemm.run(stream) != cutlass::Status::kSuccess) return fail(OZ_CUDA, "INT8 GEMM: launch", cudaGetLastError());
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return OZ_OK;
}

template <bool LMajorM, bool RMajorN>
int i8_gemm(int M, int N, int K, int L, const int8_t* Lp, int64_t ldl, int64_t batchL, const int8_t* Rp, int64_t ldr, int64_t batchR,
            int32_t* D, int64_t batchD, cudaStream_t stream) {
  // 256 x 256 tiles on SM pairs for outputs of at least 256 x 256.  Tiles that pad a 547-row block less were measured and are
  // slower: 128 x 128 on one SM 25.4 and 256 x 192 25.5 against 29.3 TFLOP/s for a 547^4 task with 211 positions.
  if (M >= 256 && N >= 256) return i8_gemm_cfg<I8Large, LMajorM, RMajorN>(M, N, K, L, Lp, ldl, batchL, Rp, ldr, batchR, D, batchD, stream);
  return i8_gemm_cfg<I8Small, LMajorM, RMajorN>(M, N, K, L, Lp, ldl, batchL, Rp, ldr, batchR, D, batchD, stream);
}

inline size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }

inline int up16(int x) { return (x + 15) & ~15; }
inline int up4(int x) { return (x + 3) & ~3; }

// workspace of a chunk of `c` items (p = 0: single product); padded extents kP, nP (16), pP (4)
struct Workspace {
  size_t qA, qX, planes, qT, qB, eA, fX, gT, hB, total;
  Workspace(int64_t c, int m, int k, int n, int p, int S) {
    const size_t kP = up16(k), nP = up16(n), pP = up4(p);
    size_t o = 0;
    auto take = [&](size_t bytes) { const size_t at = o; o += up256(bytes); return at; };
    qA = take((size_t)c * m * S * kP);
    qX = take((size_t)c * S * kP * nP);
    planes = take((size_t)c * S * 4 * m * std::max(nP, pP));
    qT = take(p ? (size_t)c * m * S * nP : 0);
    qB = take(p ? (size_t)c * pP * S * nP : 0);
    eA = take((size_t)c * m * 4); fX = take((size_t)c * nP * 4);
    gT = take(p ? (size_t)c * m * 4 : 0); hB = take(p ? (size_t)c * pP * 4 : 0);
    total = o;
  }
};

#define OZ_LAUNCH_CHECK(what)                                                    \
  do {                                                                           \
    cudaError_t e_ = cudaGetLastError();                                         \
    if (e_ != cudaSuccess) return fail(OZ_CUDA, what, e_);                       \
    g_launches.fetch_add(1, std::memory_order_relaxed);                          \
  } while (0)

// one chunk of c items; p == 0: C (m x n) = A X, else C (m x p) += alpha (A X) B^T
template <int S>
int run_chunk(int m, int k, int n, int p, int c, double alpha, const double* A, const double* X, const double* B, double* C,
              char* ws, cudaStream_t st) {
  const Workspace w(c, m, k, n, p, S);
  const int kP = up16(k), nP = up16(n), pP = up4(p);
  int8_t *qA = (int8_t*)(ws + w.qA), *qX = (int8_t*)(ws + w.qX), *qT = (int8_t*)(ws + w.qT), *qB = (int8_t*)(ws + w.qB);
  int32_t *planes = (int32_t*)(ws + w.planes), *eA = (int32_t*)(ws + w.eA), *fX = (int32_t*)(ws + w.fX), *gT = (int32_t*)(ws + w.gT),
          *hB = (int32_t*)(ws + w.hB);
  const int64_t rowsA = (int64_t)c * m;
  slice_rows_kernel<S, false><<<(unsigned)((rowsA + 7) / 8), 256, 0, st>>>(A, (int64_t)m * k, k, m, m, k, kP, rowsA, qA, eA);
  OZ_LAUNCH_CHECK("slice_rows_kernel(A) launch");
  slice_cols_kernel<S, true><<<dim3((nP + 127) / 128, c), 256, 0, st>>>(X, (int64_t)k * n, n, k, n, kP, nP, qX, fX);
  OZ_LAUNCH_CHECK("slice_cols_kernel(X) launch");
  const int64_t ps1 = (int64_t)c * m * nP;
  for (int d = 0; d < S; ++d) {                               // diagonal d: L slices 0..d, R slices d..0 = slots S-1-d..S-1
    const int rc = i8_gemm<false, true>(m, nP, (d + 1) * kP, c, qA, (int64_t)S * kP, (int64_t)m * S * kP, qX + (int64_t)(S - 1 - d) * kP * nP,
                                 nP, (int64_t)S * kP * nP, planes + d * ps1, (int64_t)m * nP, st);
    if (rc != OZ_OK) return rc;
  }
  if (p == 0) {
    const int64_t nquad = ps1 / 4;
    combine_out_kernel<S, false><<<(unsigned)std::min<int64_t>((nquad + 255) / 256, 148 * 16), 256, 0, st>>>(planes, ps1, m, n, nP, nquad, eA,
                                                                                                        fX, 1.0, C);
    OZ_LAUNCH_CHECK("combine_out_kernel launch");
    return OZ_OK;
  }
  {
    const unsigned grid = (unsigned)((rowsA + 7) / 8);
    if (nP <= 128) combine_slice_kernel<S, 1><<<grid, 256, 0, st>>>(planes, ps1, m, nP, rowsA, eA, m, fX, nP, qT, gT);
    else if (nP <= 256) combine_slice_kernel<S, 2><<<grid, 256, 0, st>>>(planes, ps1, m, nP, rowsA, eA, m, fX, nP, qT, gT);
    else if (nP <= 512) combine_slice_kernel<S, 4><<<grid, 256, 0, st>>>(planes, ps1, m, nP, rowsA, eA, m, fX, nP, qT, gT);
    else if (nP <= 1024) combine_slice_kernel<S, 8><<<grid, 256, 0, st>>>(planes, ps1, m, nP, rowsA, eA, m, fX, nP, qT, gT);
    else combine_slice_kernel<S, 0><<<grid, 256, 0, st>>>(planes, ps1, m, nP, rowsA, eA, m, fX, nP, qT, gT);
  }
  OZ_LAUNCH_CHECK("combine_slice_kernel launch");
  const int64_t rowsB = (int64_t)c * pP;
  slice_rows_kernel<S, true><<<(unsigned)((rowsB + 7) / 8), 256, 0, st>>>(B, (int64_t)p * n, n, p, pP, n, nP, rowsB, qB, hB);
  OZ_LAUNCH_CHECK("slice_rows_kernel(B) launch");
  const int64_t ps2 = (int64_t)c * m * pP;
  for (int d = 0; d < S; ++d) {
    const int rc = i8_gemm<false, false>(m, pP, (d + 1) * nP, c, qT, (int64_t)S * nP, (int64_t)m * S * nP, qB + (int64_t)(S - 1 - d) * nP,
                                  (int64_t)S * nP, (int64_t)pP * S * nP, planes + d * ps2, (int64_t)m * pP, st);
    if (rc != OZ_OK) return rc;
  }
  const int64_t nquad = ps2 / 4;
  combine_out_kernel<S, true><<<(unsigned)std::min<int64_t>((nquad + 255) / 256, 148 * 16), 256, 0, st>>>(planes, ps2, m, p, pP, nquad, gT, hB,
                                                                                                     alpha, C);
  OZ_LAUNCH_CHECK("combine_out_kernel launch");
  return OZ_OK;
}

// ---- one task of H_eff * Psi (su2_task_view): F += coef sum_pos alpha_pos Aop_pos E Dop_pos^T -----------------------------------------
// recombination of product 2 with the sum over the positions of a chunk:
//   dst[i][j] += coef sum_b alpha_b 2^(g_(b,i) + h_(b,j)) sum_d P_d[b][i][j] 2^(-W (d+2)),   b in index order (deterministic)
// planes: [S][items][rowsT][colsP]; g: [items][rowsT]; h: [items or 1][colsP] (h_pitch 0: D is the same block for all positions)
template <int S>
__global__ void __launch_bounds__(256)
combine_reduce_kernel(const int32_t* __restrict__ planes, int64_t plane_stride, int items, int rowsT, int rows, int cols, int colsP,
                      const int32_t* __restrict__ g_row, const int32_t* __restrict__ h_col, int h_pitch,
                      const double* __restrict__ alpha, double coef, double* __restrict__ dst) {
  const int cq = (cols + 3) >> 2;
  const int64_t nquad = (int64_t)rows * cq;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nquad; t += (int64_t)gridDim.x * blockDim.x) {
    const int i = (int)(t / cq), j = (int)(t - (int64_t)i * cq) * 4;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int b = 0; b < items; ++b) {
      double v[4];
      combine4<S>(planes, plane_stride, ((int64_t)b * rowsT + i) * colsP + j, v);
      const int g = g_row[(int64_t)b * rowsT + i];
      const int4 hj = *(const int4*)(h_col + (int64_t)b * h_pitch + j);
      const double a = coef * (alpha ? alpha[b] : 1.0);
      acc[0] += a * scale2(v[0], g + hj.x); acc[1] += a * scale2(v[1], g + hj.y);
      acc[2] += a * scale2(v[2], g + hj.z); acc[3] += a * scale2(v[3], g + hj.w);
    }
    double* o = dst + (int64_t)i * cols + j;
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (j + u < cols) o[u] += acc[u];
  }
}

// bytes of workspace a chunk of c positions of this task needs, and the carve-up
struct TaskSpace {
  size_t qA, qX, planes, qT, qB, eA, fX, gT, hB, total;
  int kP, nP, mP, pP, rowsT;
  TaskSpace(const su2_task_view& t, int64_t c, int S) {
    kP = up16(t.k); nP = up16(t.n); mP = up16(t.m);
    pP = t.transD ? up16(t.p) : up4(t.p);
    rowsT = t.transA ? mP : t.m;                    // an M-major left operand brings its padded rows along
    const int64_t cA = t.strideA ? c : 1, cD = t.strideD ? c : 1;
    size_t o = 0;
    auto take = [&](size_t bytes) { const size_t at = o; o += up256(bytes); return at; };
    qA = take((size_t)cA * rowsT * S * kP);
    qX = take((size_t)S * kP * nP);
    planes = take((size_t)c * S * 4 * rowsT * std::max(nP, pP));
    qT = take((size_t)c * rowsT * S * nP);
    qB = take((size_t)cD * pP * S * nP);
    eA = take((size_t)cA * rowsT * 4); fX = take((size_t)nP * 4);
    gT = take((size_t)c * rowsT * 4); hB = take((size_t)cD * pP * 4);
    total = o;
  }
};

template <int S>
int run_task(const su2_task_view& t, const double* psi, double* out, char* ws, size_t ws_bytes, cudaStream_t st) {
  if ((int64_t)S * up16(std::max(t.k, t.n)) * 127 * 127 >= ((int64_t)1 << 31)) return fail(OZ_INVALID, "task: contraction too long for exact int32 accumulation");
  int64_t c = t.npos;
  while (c > 1 && TaskSpace(t, c, S).total > ws_bytes) c = (c + 1) / 2;
  const TaskSpace w(t, c, S);
  if (w.total > ws_bytes) return fail(OZ_INVALID, "task: workspace below one position");
  const int kP = w.kP, nP = w.nP, mP = w.mP, pP = w.pP, rowsT = w.rowsT;
  int8_t *qA = (int8_t*)(ws + w.qA), *qX = (int8_t*)(ws + w.qX), *qT = (int8_t*)(ws + w.qT), *qB = (int8_t*)(ws + w.qB);
  int32_t *planes = (int32_t*)(ws + w.planes), *eA = (int32_t*)(ws + w.eA), *fX = (int32_t*)(ws + w.fX), *gT = (int32_t*)(ws + w.gT),
          *hB = (int32_t*)(ws + w.hB);
  // E is the same for every position: sliced once per task
  slice_cols_kernel<S, true><<<dim3((nP + 127) / 128, 1), 256, 0, st>>>(psi + t.e_off, 0, t.n, t.k, t.n, kP, nP, qX, fX);
  OZ_LAUNCH_CHECK("slice_cols_kernel(E) launch");
  for (int64_t pos0 = 0; pos0 < t.npos; pos0 += c) {
    const int cc = (int)std::min<int64_t>(c, t.npos - pos0);
    const int cA = t.strideA ? cc : 1, cD = t.strideD ? cc : 1;
    const double* A = t.A + pos0 * t.strideA;
    const double* D = t.D + pos0 * t.strideD;
    if (pos0 == 0 || t.strideA) {
      if (t.transA) slice_cols_kernel<S, false><<<dim3((mP + 127) / 128, cA), 256, 0, st>>>(A, t.strideA, t.ldA, t.k, t.m, kP, mP, qA, eA);
      else slice_rows_kernel<S, false><<<(unsigned)(((int64_t)cA * t.m + 7) / 8), 256, 0, st>>>(A, t.strideA, t.ldA, t.m, t.m, t.k, kP, (int64_t)cA * t.m, qA, eA);
      OZ_LAUNCH_CHECK("slice kernel (A) launch");
    }
    if (pos0 == 0 || t.strideD) {
      if (t.transD) slice_cols_kernel<S, true><<<dim3((pP + 127) / 128, cD), 256, 0, st>>>(D, t.strideD, t.ldD, t.n, t.p, nP, pP, qB, hB);
      else slice_rows_kernel<S, true><<<(unsigned)(((int64_t)cD * pP + 7) / 8), 256, 0, st>>>(D, t.strideD, t.ldD, t.p, pP, t.n, nP, (int64_t)cD * pP, qB, hB);
      OZ_LAUNCH_CHECK("slice kernel (D) launch");
    }
    const int64_t ps1 = (int64_t)cc * rowsT * nP;
    for (int d = 0; d < S; ++d) {
      int rc;
      if (t.transA) rc = i8_gemm<true, true>(rowsT, nP, (d + 1) * kP, cc, qA, mP, t.strideA ? (int64_t)S * kP * mP : 0, qX + (int64_t)(S - 1 - d) * kP * nP,
                                             nP, 0, planes + d * ps1, (int64_t)rowsT * nP, st);
      else if (t.strideA)   // E is shared and the rows of all positions are contiguous: ONE product with cc * m rows (no row padding per position)
        rc = i8_gemm<false, true>(cc * rowsT, nP, (d + 1) * kP, 1, qA, (int64_t)S * kP, 0, qX + (int64_t)(S - 1 - d) * kP * nP, nP, 0,
                                  planes + d * ps1, 0, st);
      else rc = i8_gemm<false, true>(rowsT, nP, (d + 1) * kP, cc, qA, (int64_t)S * kP, 0, qX + (int64_t)(S - 1 - d) * kP * nP, nP, 0,
                                     planes + d * ps1, (int64_t)rowsT * nP, st);
      if (rc != OZ_OK) return rc;
    }
    {
      const int64_t lines = (int64_t)cc * rowsT;
      const unsigned grid = (unsigned)((lines + 7) / 8);
      const int ep = t.strideA ? rowsT : 0;
      if (nP <= 128) combine_slice_kernel<S, 1><<<grid, 256, 0, st>>>(planes, ps1, rowsT, nP, lines, eA, ep, fX, 0, qT, gT);
      else if (nP <= 256) combine_slice_kernel<S, 2><<<grid, 256, 0, st>>>(planes, ps1, rowsT, nP, lines, eA, ep, fX, 0, qT, gT);
      else if (nP <= 512) combine_slice_kernel<S, 4><<<grid, 256, 0, st>>>(planes, ps1, rowsT, nP, lines, eA, ep, fX, 0, qT, gT);
      else if (nP <= 1024) combine_slice_kernel<S, 8><<<grid, 256, 0, st>>>(planes, ps1, rowsT, nP, lines, eA, ep, fX, 0, qT, gT);
      else combine_slice_kernel<S, 0><<<grid, 256, 0, st>>>(planes, ps1, rowsT, nP, lines, eA, ep, fX, 0, qT, gT);
      OZ_LAUNCH_CHECK("combine_slice_kernel launch");
    }
    const int64_t ps2 = (int64_t)cc * rowsT * pP;
    for (int d = 0; d < S; ++d) {
      int rc;
      if (t.transD) rc = i8_gemm<false, true>(rowsT, pP, (d + 1) * nP, cc, qT, (int64_t)S * nP, (int64_t)rowsT * S * nP,
                                              qB + (int64_t)(S - 1 - d) * nP * pP, pP, t.strideD ? (int64_t)S * nP * pP : 0, planes + d * ps2,
                                              (int64_t)rowsT * pP, st);
      else rc = i8_gemm<false, false>(rowsT, pP, (d + 1) * nP, cc, qT, (int64_t)S * nP, (int64_t)rowsT * S * nP, qB + (int64_t)(S - 1 - d) * nP,
                                      (int64_t)S * nP, t.strideD ? (int64_t)pP * S * nP : 0, planes + d * ps2, (int64_t)rowsT * pP, st);
      if (rc != OZ_OK) return rc;
    }
    const int64_t nquad = (int64_t)t.m * ((t.p + 3) / 4);
    combine_reduce_kernel<S><<<(unsigned)std::min<int64_t>((nquad + 255) / 256, 148 * 16), 256, 0, st>>>(
        planes, ps2, cc, rowsT, t.m, t.p, pP, gT, hB, t.strideD ? pP : 0, t.alpha ? t.alpha + pos0 : nullptr, t.coef, out + t.f_off);
    OZ_LAUNCH_CHECK("combine_reduce_kernel launch");
  }
  return OZ_OK;
}

int run_chunk_s(int S, int m, int k, int n, int p, int c, double alpha, const double* A, const double* X, const double* B, double* C,
                char* ws, cudaStream_t st) {
  switch (S) {
    case 2: return run_chunk<2>(m, k, n, p, c, alpha, A, X, B, C, ws, st);
    case 3: return run_chunk<3>(m, k, n, p, c, alpha, A, X, B, C, ws, st);
    case 4: return run_chunk<4>(m, k, n, p, c, alpha, A, X, B, C, ws, st);
    case 5: return run_chunk<5>(m, k, n, p, c, alpha, A, X, B, C, ws, st);
    case 6: return run_chunk<6>(m, k, n, p, c, alpha, A, X, B, C, ws, st);
    default: return run_chunk<7>(m, k, n, p, c, alpha, A, X, B, C, ws, st);
  }
}

int run(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, const double* X, const double* B, double* C, int S,
        void* workspace, size_t workspace_bytes, cudaStream_t st) {
  g_err[0] = 0;
  const bool pair = p != 0;
  if (m <= 0 || k <= 0 || n <= 0 || p < 0 || batch < 0 || !A || !X || !C || (pair && !B)) return fail(OZ_INVALID, "null pointer, non-positive dimension or negative batch");
  if (S == 0) S = OZ_SMAX;
  if (S < 2 || S > OZ_SMAX) return fail(OZ_INVALID, "nslices must be 0 or 2..7");
  if ((int64_t)S * up16(std::max(k, n)) * 127 * 127 >= ((int64_t)1 << 31)) return fail(OZ_INVALID, "contraction too long for exact int32 accumulation");
  if (((uintptr_t)A | (uintptr_t)X | (uintptr_t)B | (uintptr_t)C) & 7) return fail(OZ_INVALID, "operands must be 8-byte aligned");
  if (workspace && ((uintptr_t)workspace & 255)) return fail(OZ_INVALID, "workspace must be 256-byte aligned");
  if (batch == 0) return OZ_OK;
  if (workspace_bytes == 0) {
    if (workspace) return fail(OZ_INVALID, "workspace given without its size");
    workspace_bytes = (size_t)2 << 30;
  }
  // largest chunk that fits (the table sizes are monotone in c and at most 9 * 256 bytes above linear)
  const size_t per_item = Workspace(1, m, k, n, p, S).total;
  if (per_item > workspace_bytes) return fail(OZ_INVALID, "workspace limit below one item");
  int64_t c = std::min<int64_t>({batch, 65535, (int64_t)(workspace_bytes / per_item) + 1});
  while (c > 1 && Workspace(c, m, k, n, p, S).total > workspace_bytes) --c;
  if ((int64_t)c * m * std::max({k, n, p}) * S >= ((int64_t)1 << 40)) return fail(OZ_INVALID, "chunk too large");
  char* ws = (char*)workspace;
  if (!ws) {
    cudaError_t e = cudaMallocAsync((void**)&ws, Workspace(c, m, k, n, p, S).total, st);
    if (e != cudaSuccess) return fail(OZ_CUDA, "cudaMallocAsync(workspace)", e);
  }
  int rc = OZ_OK;
  const int pp = pair ? p : n;
  for (int64_t b0 = 0; b0 < batch && rc == OZ_OK; b0 += c) {
    const int cc = (int)std::min<int64_t>(c, batch - b0);
    rc = run_chunk_s(S, m, k, n, p, cc, alpha, A + b0 * m * k, X + b0 * k * n, pair ? B + b0 * p * n : nullptr, C + b0 * m * pp, ws, st);
  }
  if (!workspace) cudaFreeAsync(ws, st);
  return rc;
}

}  // namespace su2oz

using namespace su2oz;

extern "C" int32_t su2_gemm_pair_batched_i8(int32_t m, int32_t k, int32_t n, int32_t p, int64_t batch, double alpha, const double* A,
                                            const double* X, const double* B, double* C, int32_t nslices, void* workspace,
                                            size_t workspace_bytes, void* cuda_stream) {
  if (p <= 0) { g_err[0] = 0; return fail(OZ_INVALID, "null pointer, non-positive dimension or negative batch"); }
  return run(m, k, n, p, batch, alpha, A, X, B, C, nslices, workspace, workspace_bytes, (cudaStream_t)cuda_stream);
}

extern "C" int32_t su2_matmul_batched_i8(int32_t m, int32_t k, int32_t n, int64_t batch, const double* A, const double* X, double* C,
                                         int32_t nslices, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  return run(m, k, n, 0, batch, 1.0, A, X, nullptr, C, nslices, workspace, workspace_bytes, (cudaStream_t)cuda_stream);
}

extern "C" int32_t su2_heff_apply_i8(const su2_task_view* tasks, int64_t ntask, const double* psi, double* out, int64_t psi_len,
                                     int32_t nslices, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  g_err[0] = 0;
  if (!tasks || ntask < 0 || !psi || !out || psi == out || psi_len < 0 || !workspace || ((uintptr_t)workspace & 255))
    return fail(OZ_INVALID, "null pointer, out aliasing psi, or a workspace that is not 256-byte aligned");
  if (nslices == 0) nslices = OZ_SMAX;
  if (nslices < 2 || nslices > OZ_SMAX) return fail(OZ_INVALID, "nslices must be 0 or 2..7");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaMemsetAsync(out, 0, (size_t)psi_len * sizeof(double), st);
  if (e != cudaSuccess) return fail(OZ_CUDA, "cudaMemsetAsync(out)", e);
  for (int64_t i = 0; i < ntask; ++i) {
    const su2_task_view& t = tasks[i];
    if (!t.A || !t.D || t.m <= 0 || t.k <= 0 || t.n <= 0 || t.p <= 0 || t.npos <= 0) return fail(OZ_INVALID, "task: null operand or non-positive extent");
    int rc;
    switch (nslices) {
      case 2: rc = run_task<2>(t, psi, out, (char*)workspace, workspace_bytes, st); break;
      case 3: rc = run_task<3>(t, psi, out, (char*)workspace, workspace_bytes, st); break;
      case 4: rc = run_task<4>(t, psi, out, (char*)workspace, workspace_bytes, st); break;
      case 5: rc = run_task<5>(t, psi, out, (char*)workspace, workspace_bytes, st); break;
      case 6: rc = run_task<6>(t, psi, out, (char*)workspace, workspace_bytes, st); break;
      default: rc = run_task<7>(t, psi, out, (char*)workspace, workspace_bytes, st); break;
    }
    if (rc != OZ_OK) return rc;
  }
  return OZ_OK;
}

extern "C" size_t su2_ozaki_workspace_bytes(int32_t m, int32_t k, int32_t n, int32_t p, int64_t items, int32_t nslices) {
  if (m <= 0 || k <= 0 || n <= 0 || p < 0 || items <= 0) return 0;
  if (nslices == 0) nslices = OZ_SMAX;
  if (nslices < 2 || nslices > OZ_SMAX) return 0;
  return Workspace(items, m, k, n, p, nslices).total;
}

extern "C" int64_t su2_ozaki_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

extern "C" const char* su2_ozaki_last_error(void) { return g_err; }
