// Row a4 of SURVEY section 8 in the small-block regime (every block sector of the bond holds at most
// SMALL_MAX_DIM multiplets; BASELINE.json configs[0] and configs[1]): the fused GEMM pair
//     F_s (m x p) += coef * sum_pos alpha_pos * A_pos (m x k) E_s' (k x n) D_pos^T (n x p)      (Eq. 2/3)
// on the same plan tables (DevTask / DevUnit / DevWork) as heff_dmma_kernel, with a CTA shape made for blocks of a
// few dozen doubles instead of 128 x 144 register tiles:
//   * one CTA owns a WHOLE output sector of one segment; its m8n8 DMMA accumulator tiles are dealt round-robin to
//     the warps and stay in registers over all tasks and positions of the work item (the sum over positions is the
//     K loop of the second product: the paper's stripe trick);
//   * a step (one position of one task) is a few dozen DMMAs per warp, far less than one trip to L2, so the
//     kernel lives on residency: work items are sorted into size classes DM8 = 8, 16, ..., 48 (largest of m, k,
//     n, p over the item's tasks, rounded up to 8), one launch per class with four shared tiles (A, D, E, T) of
//     DM8 x (DM8 + 4) doubles and 1, 4 or 8 warps: 3 KB (16 CTAs per SM) up to 80 KB (2 CTAs per SM);
//   * the (task, position) steps of an item form one flat sequence; inside a CTA, A and E of the next step are
//     copied (cp.async, 16-byte where alignment allows, zero fill for the pads) under the second product of the
//     current one and D under the next first product, with two CTA barriers per step; the task record of the
//     next step is fetched one step ahead; T = coef alpha_pos A_pos E goes through shared memory only;
//   * adjoint rows read the stored block transposed by swapping the two fragment strides, no extra copy.
// Work items are pulled from the plan's longest-first queue with one atomic counter; every output element is
// written by exactly one CTA (partials + reduce_kernel for split sectors): deterministic, no data atomics.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "su2_internal.h"

namespace su2 {

namespace {

__host__ __device__ inline int hs_ld(int x) { return ((x + 3) & ~7) + 4; }   // >= x, = 4 (mod 8): conflict-free fragments

__device__ __forceinline__ void hs_cp8(double* dst, const double* src, bool valid) {
  const int sz = valid ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void hs_cp16(double* dst, const double* src, bool valid) {
  const int sz = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void hs_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void hs_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void hs_dmma(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// K loop of one product for a warp that owns NR x NC m8n8 tiles: straight-line per (NR, NC), no predicated
// DMMAs (a predicated-off DMMA still takes its slot in the FP64 tensor pipe).  ap / bp: this lane's fragment
// element of tile row 0 / tile column 0 at k = 0; a_i / b_j: distance to the next owned tile; a_k / b_k: per k4 step.
template <int NR, int NC, int TRM, int TCM>
__device__ __forceinline__ void hs_mma_loop(double (&acc)[TRM][TCM][2], const double* ap, int a_i, int a_k,
                                            const double* bp, int b_j, int b_k, int ksteps) {
#pragma unroll 2
  for (int s = 0; s < ksteps; ++s) {
    double a[NR], b[NC];
#pragma unroll
    for (int i = 0; i < NR; ++i) a[i] = ap[i * a_i];
#pragma unroll
    for (int j = 0; j < NC; ++j) b[j] = bp[j * b_j];
#pragma unroll
    for (int i = 0; i < NR; ++i)
#pragma unroll
      for (int j = 0; j < NC; ++j) hs_dmma(acc[i][j], a[i], b[j]);
    ap += a_k;
    bp += b_k;
  }
}

// nr x nc of the warp's TRM x TCM tile slots exist (prefixes): pick the straight-line instance.
template <int TRM, int TCM>
__device__ __forceinline__ void hs_mma(double (&acc)[TRM][TCM][2], int nr, int nc, const double* ap, int a_i, int a_k,
                                       const double* bp, int b_j, int b_k, int ksteps) {
#define HS_CASE(R, C)                                                                                              \
  if (R <= TRM && C <= TCM && nr == R && nc == C)                                                                    \
    hs_mma_loop<(R <= TRM ? R : 1), (C <= TCM ? C : 1), TRM, TCM>(acc, ap, a_i, a_k, bp, b_j, b_k, ksteps);
  HS_CASE(1, 1) HS_CASE(1, 2) HS_CASE(2, 1) HS_CASE(2, 2) HS_CASE(3, 1) HS_CASE(3, 2)
#undef HS_CASE
  static_assert(TRM <= 3 && TCM <= 2, "add HS_CASE lines");
}

struct Step { int u, pos; };

}  // namespace


// Size class DM8 (largest dimension of any task of the item, rounded up to 8); WR x WC warps per CTA, warp
// (wr, wc) owns the m8n8 tiles (wr + WR i, wc + WC j): the A fragment of a tile row is shared by its TCM column
// tiles and the B fragment of a tile column by its TRM row tiles (5 fragment loads per 6 DMMAs at 48 x 48).
// Shared memory: four tiles of DM8 x hs_ld(DM8) doubles: A, D, E, T.  Only E carries true zeros in its pads
// (rows k..K4, columns n..N8): they annihilate whatever finite numbers earlier steps left in the pads of A and
// D, and make the pad columns of T exact zeros.
template <int DM8, int WR, int WC, int MINB>
__global__ void __launch_bounds__(32 * WR * WC, MINB)
heff_small_kernel(const DevWork* __restrict__ work, int nwork, const DevUnit* __restrict__ units,
                  const DevTask* __restrict__ tasks, const double* __restrict__ psi, double* __restrict__ out,
                  double* __restrict__ partial, int* __restrict__ counter) {
  constexpr int WARPS = WR * WC, THREADS = 32 * WARPS;
  constexpr int TRM = (DM8 / 8 + WR - 1) / WR, TCM = (DM8 / 8 + WC - 1) / WC;   // tiles per warp: rows x columns
  constexpr int LD = ((DM8 + 3) & ~7) + 4, SZ = DM8 * LD;
  extern __shared__ __align__(16) double smem[];
  __shared__ int s_item;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wr = warp % WR, wc = warp / WR;
  const int fr = lane >> 2, fc = lane & 3;
  double* const As = smem;
  double* const Ds = smem + SZ;
  double* const Es = smem + 2 * SZ;
  double* const Ts = smem + 3 * SZ;
  for (int e = tid; e < 4 * SZ; e += THREADS) smem[e] = 0.0;   // whatever sits in a pad must be finite

  // stored rows x cols block (leading dimension lds) -> shared rows of stride LD, one warp per row; pads untouched
  auto copy_rows = [&](double* dst, const double* __restrict__ src, int rows, int cols, int lds) {
    uint32_t d = (uint32_t)__cvta_generic_to_shared(dst) + (uint32_t)(warp * LD) * 8u;
    const double* s = src + (int64_t)warp * lds;
    const int64_t s_step = (int64_t)WARPS * lds;
    if (!(cols & 1) && !(lds & 1) && !((uintptr_t)src & 15)) {
      if (2 * lane < cols) {
        d += 16u * lane; s += 2 * lane;
        for (int r = warp; r < rows; r += WARPS, d += WARPS * LD * 8, s += s_step)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(s) : "memory");
      }
    } else {
      d += 8u * lane; s += lane;
      const bool on0 = lane < cols, on1 = DM8 > 32 && lane + 32 < cols;
      for (int r = warp; r < rows; r += WARPS, d += WARPS * LD * 8, s += s_step) {
        if (on0) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(s) : "memory");
        if (on1) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d + 256u), "l"(s + 32) : "memory");
      }
    }
  };
  // E: the same with zero fill up to rows_pad x cols_pad
  auto copy_e = [&](const double* __restrict__ src, int rows, int cols, int lde, int rows_pad, int cols_pad) {
    for (int r = warp; r < rows_pad; r += WARPS)
      for (int c = lane; c < cols_pad; c += 32) {
        const bool valid = r < rows && c < cols;
        hs_cp8(Es + r * LD + c, valid ? src + (int64_t)r * lde + c : src, valid);
      }
  };
  auto issue_AE = [&](const DevTask& t, int pos, bool with_e) {
    const double* A = t.A + (int64_t)pos * t.strideA;
    if (t.flags & TASK_TRANS_A) copy_rows(As, A, t.k, t.m, t.ldA);
    else copy_rows(As, A, t.m, t.k, t.ldA);
    if (with_e) copy_e(psi + t.e_off, t.k, t.n, t.ldE, (t.k + 3) & ~3, (t.n + 7) & ~7);
  };
  auto issue_D = [&](const DevTask& t, int pos) {
    const double* D = t.D + (int64_t)pos * t.strideD;
    if (t.flags & TASK_TRANS_D) copy_rows(Ds, D, t.n, t.p, t.ldD);
    else copy_rows(Ds, D, t.p, t.n, t.ldD);
  };

  for (;;) {
    __syncthreads();                       // previous item (and the zero fill) done with shared memory
    if (tid == 0) s_item = atomicAdd(counter, 1);
    __syncthreads();
    const int item = s_item;
    if (item >= nwork) break;
    const DevWork w = work[item];
    const int M8 = (w.m + 7) & ~7, P8 = (w.p + 7) & ~7;
    // tile rows / tile columns of F this warp owns (prefixes of its TRM x TCM slots; warp-uniform)
    const int nr = min(TRM, max(0, (M8 / 8 - wr + WR - 1) / WR)), np = min(TCM, max(0, (P8 / 8 - wc + WC - 1) / WC));
    double acc[TRM][TCM][2];
#pragma unroll
    for (int i = 0; i < TRM; ++i)
#pragma unroll
      for (int j = 0; j < TCM; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    DevUnit un = units[w.unit0];
    DevTask tc = tasks[un.task];
    Step cur{w.unit0, un.pos0};
    double scale = tc.coef * (tc.alpha ? tc.alpha[cur.pos] : 1.0);
    issue_AE(tc, cur.pos, true);
    hs_commit();
    hs_wait<0>();
    __syncthreads();
    issue_D(tc, cur.pos);
    hs_commit();
    while (cur.u < w.unit1) {
      // next step and its task record (in flight under the first product)
      Step nxt{cur.u, cur.pos + 1};
      DevUnit un_n = un;
      const bool new_unit = nxt.pos >= un.pos1;
      if (new_unit) {
        nxt.u = cur.u + 1;
        if (nxt.u < w.unit1) { un_n = units[nxt.u]; nxt.pos = un_n.pos0; }
      }
      const bool has_next = nxt.u < w.unit1;
      DevTask tn = tc;
      if (new_unit && has_next) tn = tasks[un_n.task];

      const int K4 = (tc.k + 3) & ~3, N8 = (tc.n + 7) & ~7;
      // fragment strides: element (row r, inner index j) of the operand sits at r * sr + j * sc
      const int a_sr = (tc.flags & TASK_TRANS_A) ? 1 : LD, a_sc = (tc.flags & TASK_TRANS_A) ? LD : 1;
      const int d_sr = (tc.flags & TASK_TRANS_D) ? 1 : LD, d_sc = (tc.flags & TASK_TRANS_D) ? LD : 1;

      // ---- first product: T = scale * A E
      {
        const int nn = min(TCM, max(0, (N8 / 8 - wc + WC - 1) / WC));
        double tacc[TRM][TCM][2];
#pragma unroll
        for (int i = 0; i < TRM; ++i)
#pragma unroll
          for (int j = 0; j < TCM; ++j) tacc[i][j][0] = tacc[i][j][1] = 0.0;
        hs_mma<TRM, TCM>(tacc, nr, nn, As + (8 * wr + fr) * a_sr + fc * a_sc, 8 * WR * a_sr, 4 * a_sc,
                         Es + fc * LD + 8 * wc + fr, 8 * WC, 4 * LD, K4 >> 2);
#pragma unroll
        for (int i = 0; i < TRM; ++i)
#pragma unroll
          for (int j = 0; j < TCM; ++j)
            if (i < nr && j < nn)
              *reinterpret_cast<double2*>(Ts + (8 * (wr + WR * i) + fr) * LD + 8 * (wc + WC * j) + 2 * fc) =
                  make_double2(scale * tacc[i][j][0], scale * tacc[i][j][1]);
      }
      hs_wait<0>();                        // D of this step
      __syncthreads();                     // T and D visible; A and E free
      if (has_next) {
        issue_AE(tn, nxt.pos, new_unit);
        scale = tn.coef * (tn.alpha ? tn.alpha[nxt.pos] : 1.0);
      }
      hs_commit();
      // ---- second product: F += T D^T, K = n (padded to 8)
      hs_mma<TRM, TCM>(acc, nr, np, Ts + (8 * wr + fr) * LD + fc, 8 * WR * LD, 4,
                       Ds + (8 * wc + fr) * d_sr + fc * d_sc, 8 * WC * d_sr, 4 * d_sc, N8 >> 2);
      hs_wait<0>();                        // A (and E) of the next step
      __syncthreads();                     // ... visible; T and D free
      if (has_next) issue_D(tn, nxt.pos);
      hs_commit();
      cur = nxt; un = un_n; tc = tn;
    }
    hs_wait<0>();

    // ---- write the sector: plain store, or += for the accumulate flag
    double* dst = ((w.to_partial & 1) ? partial : out) + w.dst_off;
#pragma unroll
    for (int i = 0; i < TRM; ++i)
#pragma unroll
      for (int j = 0; j < TCM; ++j) {
        const int r = 8 * (wr + WR * i) + fr, c = 8 * (wc + WC * j) + 2 * fc;
        if (i < nr && j < np && r < w.m) {
          double* q = dst + (int64_t)r * w.ldo + c;
          if (w.to_partial & 2) {
            if (c < w.p) q[0] += acc[i][j][0];
            if (c + 1 < w.p) q[1] += acc[i][j][1];
          } else {
            if (c < w.p) q[0] = acc[i][j][0];
            if (c + 1 < w.p) q[1] = acc[i][j][1];
          }
        }
      }
  }
}

namespace {

template <int DM8, int WR, int WC, int MINB>
su2_status launch_class(const su2_plan* plan, int cls, const double* psi, double* out, double* partial, cudaStream_t stream) {
  const int begin = plan->small_begin[cls], nwork = plan->small_begin[cls + 1] - begin;
  if (nwork <= 0) return SU2_OK;
  const size_t smem = sizeof(double) * 4 * (size_t)DM8 * hs_ld(DM8);
  constexpr int WARPS = WR * WC;
  auto kern = heff_small_kernel<DM8, WR, WC, MINB>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) { set_cuda_error("cudaFuncSetAttribute(heff_small_kernel)", (int)e); return SU2_ERR_CUDA; }
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 32 * WARPS, smem);
  if (e != cudaSuccess || per_sm < 1) { set_cuda_error("occupancy(heff_small_kernel)", (int)e); return SU2_ERR_CUDA; }
  const int grid = std::min(nwork, plan->num_sms * per_sm);
  kern<<<grid, 32 * WARPS, smem, stream>>>(plan->d_work + begin, nwork, plan->d_units, plan->d_tasks, psi, out, partial,
                                           plan->d_counter + cls);
  e = cudaGetLastError();
  if (e != cudaSuccess) { set_cuda_error("heff_small_kernel launch", (int)e); return SU2_ERR_CUDA; }
  count_launch();
  return SU2_OK;
}

}  // namespace

// One launch per non-empty size class, largest blocks first; plan->d_counter[0..5] must be zero.
su2_status launch_heff_small(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  su2_status st;
  if ((st = launch_class<48, 2, 4, 2>(plan, 5, psi, out, partial, stream)) != SU2_OK) return st;
  if ((st = launch_class<40, 2, 4, 3>(plan, 4, psi, out, partial, stream)) != SU2_OK) return st;
  if ((st = launch_class<32, 2, 2, 6>(plan, 3, psi, out, partial, stream)) != SU2_OK) return st;
  if ((st = launch_class<24, 2, 2, 8>(plan, 2, psi, out, partial, stream)) != SU2_OK) return st;
  if ((st = launch_class<16, 2, 2, 8>(plan, 1, psi, out, partial, stream)) != SU2_OK) return st;
  return launch_class<8, 1, 1, 16>(plan, 0, psi, out, partial, stream);
}

}  // namespace su2
