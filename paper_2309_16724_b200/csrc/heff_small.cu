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

// Stored dense row-major rows x cols -> shared tile (leading dimension ld), zero-filled up to rows_pad x cols_pad.
template <int VEC, int HS_THREADS>
__device__ __forceinline__ void hs_copy(double* __restrict__ dst, int ld, const double* __restrict__ src, int rows, int cols,
                                        int rows_pad, int cols_pad, int tid) {
  const int cv = cols_pad / VEC;               // copies per padded row (cols_pad is a multiple of 4)
  const int total = rows_pad * cv;
  int r = tid / cv, c = tid - r * cv;
  const int dr = HS_THREADS / cv, dc = HS_THREADS - dr * cv;
  for (int e = tid; e < total; e += HS_THREADS) {
    const bool valid = r < rows && VEC * c < cols;
    const double* s = valid ? src + (int64_t)r * cols + VEC * c : src;
    if (VEC == 2) hs_cp16(dst + r * ld + 2 * c, s, valid);
    else hs_cp8(dst + r * ld + c, s, valid);
    r += dr; c += dc;
    if (c >= cv) { c -= cv; ++r; }
  }
}

template <int HS_THREADS>
__device__ __forceinline__ void hs_copy_any(double* dst, int ld, const double* src, int rows, int cols, int rows_pad,
                                            int cols_pad, int tid) {
  if (!(cols & 1) && !((uintptr_t)src & 15)) hs_copy<2, HS_THREADS>(dst, ld, src, rows, cols, rows_pad, cols_pad, tid);
  else hs_copy<1, HS_THREADS>(dst, ld, src, rows, cols, rows_pad, cols_pad, tid);
}

struct Step { int u, pos; };

}  // namespace


// Size class DM8 (largest dimension of any task of the item, rounded up to 8), WARPS warps per CTA.
// Shared memory: four tiles of DM8 x hs_ld(DM8) doubles: A, D, E, T.
template <int DM8, int WARPS>
__global__ void __launch_bounds__(32 * WARPS)
heff_small_kernel(const DevWork* __restrict__ work, int nwork, const DevUnit* __restrict__ units,
                  const DevTask* __restrict__ tasks, const double* __restrict__ psi, double* __restrict__ out,
                  double* __restrict__ partial, int* __restrict__ counter) {
  constexpr int THREADS = 32 * WARPS;
  constexpr int MAXT = ((DM8 / 8) * (DM8 / 8) + WARPS - 1) / WARPS;   // m8n8 tiles per warp
  constexpr int LD = ((DM8 + 3) & ~7) + 4, SZ = DM8 * LD;
  extern __shared__ __align__(16) double smem[];
  __shared__ int s_item;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int fr = lane >> 2, fc = lane & 3;
  double* const As = smem;
  double* const Ds = smem + SZ;
  double* const Es = smem + 2 * SZ;
  double* const Ts = smem + 3 * SZ;
  for (int e = tid; e < 4 * SZ; e += THREADS) smem[e] = 0.0;   // stale pads must at least be finite

  auto issue_AE = [&](const DevTask& t, int pos, bool with_e) {
    const int M8 = (t.m + 7) & ~7, K4 = (t.k + 3) & ~3, N8 = (t.n + 7) & ~7;
    const double* A = t.A + (int64_t)pos * t.strideA;
    if (t.flags & TASK_TRANS_A) hs_copy_any<THREADS>(As, LD, A, t.k, t.m, K4, M8, tid);
    else hs_copy_any<THREADS>(As, LD, A, t.m, t.k, M8, K4, tid);
    if (with_e) hs_copy_any<THREADS>(Es, LD, psi + t.e_off, t.k, t.n, K4, N8, tid);
  };
  auto issue_D = [&](const DevTask& t, int pos) {
    const int N8 = (t.n + 7) & ~7, P8 = (t.p + 7) & ~7;
    const double* D = t.D + (int64_t)pos * t.strideD;
    if (t.flags & TASK_TRANS_D) hs_copy_any<THREADS>(Ds, LD, D, t.n, t.p, N8, P8, tid);
    else hs_copy_any<THREADS>(Ds, LD, D, t.p, t.n, P8, N8, tid);
  };

  for (;;) {
    __syncthreads();                       // previous item (and the zero fill) done with shared memory
    if (tid == 0) s_item = atomicAdd(counter, 1);
    __syncthreads();
    const int item = s_item;
    if (item >= nwork) break;
    const DevWork w = work[item];
    const int pt = (w.p + 7) >> 3, ntile2 = ((w.m + 7) >> 3) * pt;
    double acc[MAXT][2];
#pragma unroll
    for (int i = 0; i < MAXT; ++i) acc[i][0] = acc[i][1] = 0.0;

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

      // ---- first product: T = scale * A E, m8n8 tiles dealt round-robin
      {
        const int nt = N8 >> 3, ntile1 = ((tc.m + 7) >> 3) * nt;
        double tacc[MAXT][2];
        int aoff[MAXT], eoff[MAXT];
#pragma unroll
        for (int i = 0; i < MAXT; ++i) {
          const int tl = warp + WARPS * i, tr = tl / nt, tcn = tl - tr * nt;
          tacc[i][0] = tacc[i][1] = 0.0;
          aoff[i] = (8 * tr + fr) * a_sr + fc * a_sc;
          eoff[i] = fc * LD + 8 * tcn + fr;
        }
        for (int k0 = 0; k0 < K4; k0 += 4) {
#pragma unroll
          for (int i = 0; i < MAXT; ++i)
            if (warp + WARPS * i < ntile1) hs_dmma(tacc[i], As[aoff[i] + k0 * a_sc], Es[eoff[i] + k0 * LD]);
        }
#pragma unroll
        for (int i = 0; i < MAXT; ++i) {
          const int tl = warp + WARPS * i, tr = tl / nt, tcn = tl - tr * nt;
          if (tl < ntile1)
            *reinterpret_cast<double2*>(Ts + (8 * tr + fr) * LD + 8 * tcn + 2 * fc) = make_double2(scale * tacc[i][0], scale * tacc[i][1]);
        }
      }
      hs_wait<0>();                        // D of this step
      __syncthreads();                     // T and D visible; A and E free
      if (has_next) {
        issue_AE(tn, nxt.pos, new_unit);
        scale = tn.coef * (tn.alpha ? tn.alpha[nxt.pos] : 1.0);
      }
      hs_commit();
      // ---- second product: F += T D^T, K = n (padded to 8)
      {
        int toff[MAXT], doff[MAXT];
#pragma unroll
        for (int i = 0; i < MAXT; ++i) {
          const int tl = warp + WARPS * i, tr = tl / pt, tcn = tl - tr * pt;
          toff[i] = (8 * tr + fr) * LD + fc;
          doff[i] = (8 * tcn + fr) * d_sr + fc * d_sc;
        }
        for (int k0 = 0; k0 < N8; k0 += 4) {
#pragma unroll
          for (int i = 0; i < MAXT; ++i)
            if (warp + WARPS * i < ntile2) hs_dmma(acc[i], Ts[toff[i] + k0], Ds[doff[i] + k0 * d_sc]);
        }
      }
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
    for (int i = 0; i < MAXT; ++i) {
      const int tl = warp + WARPS * i, tr = tl / pt, tcn = tl - tr * pt;
      const int r = 8 * tr + fr, c = 8 * tcn + 2 * fc;
      if (tl < ntile2 && r < w.m) {
        double* q = dst + (int64_t)r * w.p + c;
        if (w.to_partial & 2) {
          if (c < w.p) q[0] += acc[i][0];
          if (c + 1 < w.p) q[1] += acc[i][1];
        } else {
          if (c < w.p) q[0] = acc[i][0];
          if (c + 1 < w.p) q[1] = acc[i][1];
        }
      }
    }
  }
}

namespace {

template <int DM8, int WARPS>
su2_status launch_class(const su2_plan* plan, int cls, const double* psi, double* out, double* partial, cudaStream_t stream) {
  const int begin = plan->small_begin[cls], nwork = plan->small_begin[cls + 1] - begin;
  if (nwork <= 0) return SU2_OK;
  const size_t smem = sizeof(double) * 4 * (size_t)DM8 * hs_ld(DM8);
  auto kern = heff_small_kernel<DM8, WARPS>;
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
  if ((st = launch_class<48, 8>(plan, 5, psi, out, partial, stream)) != SU2_OK) return st;
  if ((st = launch_class<40, 8>(plan, 4, psi, out, partial, stream)) != SU2_OK) return st;
  if ((st = launch_class<32, 4>(plan, 3, psi, out, partial, stream)) != SU2_OK) return st;
  if ((st = launch_class<24, 4>(plan, 2, psi, out, partial, stream)) != SU2_OK) return st;
  if ((st = launch_class<16, 4>(plan, 1, psi, out, partial, stream)) != SU2_OK) return st;
  return launch_class<8, 1>(plan, 0, psi, out, partial, stream);
}

}  // namespace su2
