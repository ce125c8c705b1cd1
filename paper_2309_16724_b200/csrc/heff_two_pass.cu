// Two-pass route of H_eff * Psi (row a4 of SURVEY.md section 8; plan flag SU2_PLAN_TWO_PASS, the default of large-block bonds): the task
//     F_s (m x p) += coef sum_pos alpha_pos Aop_pos (m x k) E_s' (k x n) Dop_pos^T (n x p)          (Eq. (3))
// executed the way the paper does it (a strided-batched GEMM per product, the sum over positions as the
// inner dimension of the second one -- the "stripe" trick), but with both products on this library's own
// TMA-fed DMMA.8x8x4 GEMM and the intermediate T in a scratch that belongs to the plan (allocated by it or handed in by the caller):
//   pass 1:  T_pos = coef alpha_pos Aop_pos E           for every position of a slice        (order 1: T_pos = coef alpha_pos E Dop_pos^T)
//   pass 2:  partial[chunk] = sum_{pos in chunk} T_pos Dop_pos^T   (K loop over (pos, n))     (order 1: sum_pos Aop_pos T_pos)
//   reduce:  F_s += partial slabs in index order (deterministic, no atomics; row a5)
// Why: on sm_100a what decides DMMA throughput is the register tile of a warp and the number of independent CTAs per SM
// (profiles/r02_cfg5_shapes.md, r02_two_pass_route.md): four warps of 32 x 64, two CTAs per SM reach 90-95 % of the pipe, the
// fused kernel (heff_tma.cu: both products' accumulators in registers, T chunk in shared memory, one CTA per SM) 79 %.  T costs
// 16 bytes of HBM traffic per entry against 2 (k + p) flops.
//
// One kernel serves both passes (tp_gemm_kernel): D (M x N) = scale * sum_pos L_pos (M x K) R_pos (K x N), CTA tile 64 x 128,
// k stages of 20 staged by one elected thread with bulk-tensor copies (true extents in the tensor maps: ragged edges and the
// k tail arrive as zeros), 4 consumer warps (2 x 2).  Ragged last row / column tiles run a narrower instantiation
// (warp tile 8 NI x 8 NJ) instead of multiplying zeros.  A CTA works through several consecutive items with its pipeline kept
// full; only the producer thread reads the tables and hands the item descriptors to the consumers through shared memory.
// su2_gemm_pair_batched (gemm_two_pass.cu) runs on the same kernel with the batch items in the place of the positions.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstdio>

#include "su2_internal.h"

namespace su2 {

namespace {

constexpr int TP_NS = 3;                                   // pipeline stages
constexpr int TP_CONSUMERS = 4, TP_THREADS = 32 * (TP_CONSUMERS + 1);
constexpr int TP_LBOX_K = TP_TM * TP_KS;                   // L as stored (rows x k, pitch 20)
constexpr int TP_LBOX_M = TP_KS * TP_LLD;                  // L read transposed (k x rows, pitch 68)
constexpr int TP_LREG = TP_LBOX_M > TP_LBOX_K ? TP_LBOX_M : TP_LBOX_K;
constexpr int TP_RBOX_K = TP_TN * TP_KS;                   // R with k contiguous (columns x k, pitch 20)
constexpr int TP_RBOX_N = TP_KS * TP_RLD;                  // R with the columns contiguous (k x columns, pitch 132)
constexpr int TP_RREG = TP_RBOX_N > TP_RBOX_K ? TP_RBOX_N : TP_RBOX_K;
constexpr int TP_STAGE = TP_LREG + TP_RREG;
static_assert(TP_LREG % 16 == 0 && TP_STAGE % 16 == 0, "boxes land on 128-byte boundaries");
constexpr size_t TP_SMEM = (size_t)TP_NS * TP_STAGE * sizeof(double);

__device__ __forceinline__ unsigned tp_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void tp_mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(tp_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void tp_mbar_arrive(uint64_t* bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(tp_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tp_mbar_expect(uint64_t* bar, unsigned bytes) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"(tp_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tp_mbar_wait(uint64_t* bar, int parity) {
  unsigned ok = 0;
  while (!ok)
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(ok) : "r"(tp_smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tp_tma_box(unsigned dst, const void* map, int c0, int c1, int c2, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n"
               ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(tp_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tp_dmma(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// What one CTA does, decoded from its slice by every thread.
struct TpItem {
  const CUtensorMap *mapL, *mapR;
  int M, N, K;              // extents of the product
  int row0, col0;           // tile origin
  int npl;                  // positions summed by this item (pass 1: one)
  int lt, rn;               // L read transposed; R with the columns contiguous
  int l_row, l_row_step;    // L row coordinate offset of the first position and its step per position (T as L)
  int l_item, l_item_step;  // third coordinate of the L boxes
  int r_k, r_k_step;        // R k-coordinate offset (T as R)
  int r_item, r_item_step;
  int ni, nj;               // warp tile: 8 ni rows x 8 nj columns
  double* dst;
  int ldd;
  int acc_init;             // 1: the accumulators start from dst (dst += ...), 0: from zero
  double scale;
};

// consumer warp (wr, wc) of a 2 x 2 grid: rows [8 NI wr, +8 NI) x columns [8 NJ wc, +8 NJ) of the CTA tile
template <int NI, int NJ, bool LT, bool RN>
__device__ __forceinline__ void tp_consume(const TpItem& it, const double* __restrict__ smem, uint64_t* full, uint64_t* empty, int warp, int lane, int& step) {
  const int wr = warp >> 1, wc = warp & 1;
  const int g = lane >> 2, t = lane & 3;
  double acc[NI][NJ][2];
#pragma unroll
  for (int i = 0; i < NI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  if (it.acc_init) {   // dst += ...: start from the old values (fetched while the pipeline fills) instead of adding them at the end
    const int cb = it.col0 + wc * 8 * NJ + 2 * t, rb = it.row0 + wr * 8 * NI + g;
    if (!(it.ldd & 1) && !((uintptr_t)it.dst & 15) && rb + 8 * (NI - 1) < it.M && cb + 8 * (NJ - 1) + 1 < it.N) {
      const double* __restrict__ o = it.dst + (int64_t)rb * it.ldd + cb;   // the whole share inside the output: plain 16-byte loads
      const int64_t rstep = (int64_t)8 * it.ldd;
#pragma unroll
      for (int i = 0; i < NI; ++i, o += rstep)
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
          const double2 v = *(const double2*)(o + 8 * j);
          acc[i][j][0] = v.x; acc[i][j][1] = v.y;
        }
    } else {
#pragma unroll
      for (int i = 0; i < NI; ++i) {
        const int r = rb + i * 8;
        if (r >= it.M) continue;
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
          const int c = cb + j * 8;
          const double* o = it.dst + (int64_t)r * it.ldd + c;
          if (!(it.ldd & 1) && !((uintptr_t)it.dst & 15) && c + 1 < it.N) {
            const double2 v = *(const double2*)o;
            acc[i][j][0] = v.x; acc[i][j][1] = v.y;
          } else {
            if (c < it.N) acc[i][j][0] = o[0];
            if (c + 1 < it.N) acc[i][j][1] = o[1];
          }
        }
      }
    }
  }
  constexpr int LI = LT ? 8 : 8 * TP_KS, LS = LT ? 4 * TP_LLD : 4;          // element steps: next m8 tile, next k4 sub-step
  constexpr int RJ = RN ? 8 : 8 * TP_KS, RS = RN ? 4 * TP_RLD : 4;
  const int l_off = LT ? t * TP_LLD + wr * 8 * NI + g : (wr * 8 * NI + g) * TP_KS + t;
  const int r_off = TP_LREG + (RN ? t * TP_RLD + wc * 8 * NJ + g : (wc * 8 * NJ + g) * TP_KS + t);
  const int nsteps = (it.K + TP_KS - 1) / TP_KS;
  const int nsub_last = (it.K - (nsteps - 1) * TP_KS + 3) >> 2;            // k4 sub-steps of the last stage that hold data
  for (int pl = 0; pl < it.npl; ++pl)
    for (int s = 0; s < nsteps; ++s, ++step) {
      const int b = step % TP_NS;
      tp_mbar_wait(&full[b], (step / TP_NS) & 1);
      const double* __restrict__ st = smem + (size_t)b * TP_STAGE;
      if (s != nsteps - 1 || nsub_last == TP_KS / 4) {
        // full stage: straight-line, the fragments of sub-step + 1 are fetched before the DMMAs of this one are issued
        double af[2][NI], bf[2][NJ];
#pragma unroll
        for (int i = 0; i < NI; ++i) af[0][i] = st[l_off + i * LI];
#pragma unroll
        for (int j = 0; j < NJ; ++j) bf[0][j] = st[r_off + j * RJ];
#pragma unroll
        for (int sub = 0; sub < TP_KS / 4; ++sub) {
          const int cur = sub & 1, nxt = cur ^ 1;
          if (sub + 1 < TP_KS / 4) {
#pragma unroll
            for (int i = 0; i < NI; ++i) af[nxt][i] = st[l_off + i * LI + (sub + 1) * LS];
#pragma unroll
            for (int j = 0; j < NJ; ++j) bf[nxt][j] = st[r_off + j * RJ + (sub + 1) * RS];
          }
#pragma unroll
          for (int j = 0; j < NJ; ++j)
#pragma unroll
            for (int i = 0; i < NI; ++i) tp_dmma(acc[i][j], af[cur][i], bf[cur][j]);
        }
      } else {
        // ragged last stage of a position: only the k4 sub-steps that hold data (the rest of the box is zero fill)
#pragma unroll 1
        for (int sub = 0; sub < nsub_last; ++sub) {
          double af[NI], bf[NJ];
#pragma unroll
          for (int i = 0; i < NI; ++i) af[i] = st[l_off + i * LI + sub * LS];
#pragma unroll
          for (int j = 0; j < NJ; ++j) bf[j] = st[r_off + j * RJ + sub * RS];
#pragma unroll
          for (int j = 0; j < NJ; ++j)
#pragma unroll
            for (int i = 0; i < NI; ++i) tp_dmma(acc[i][j], af[i], bf[j]);
        }
      }
      __syncwarp();
      if (lane == 0) tp_mbar_arrive(&empty[b]);
    }
  // epilogue: dst = scale * acc (accumulator layout: row g, columns 2t, 2t + 1 of every m8n8 tile)
  const bool vec = !(it.ldd & 1) && !((uintptr_t)it.dst & 15);
  const int cbase = it.col0 + wc * 8 * NJ + 2 * t;
  const int rbase = it.row0 + wr * 8 * NI + g;
  if (vec && rbase + 8 * (NI - 1) < it.M && cbase + 8 * (NJ - 1) + 1 < it.N) {
    // this thread's whole share lies inside the output (every tile but the ragged last ones): plain 16-byte stores
    double* __restrict__ o = it.dst + (int64_t)rbase * it.ldd + cbase;
    const int64_t rstep = (int64_t)8 * it.ldd;
#pragma unroll
    for (int i = 0; i < NI; ++i, o += rstep)
#pragma unroll
      for (int j = 0; j < NJ; ++j) *(double2*)(o + 8 * j) = make_double2(it.scale * acc[i][j][0], it.scale * acc[i][j][1]);
    return;
  }
#pragma unroll
  for (int i = 0; i < NI; ++i) {
    const int r = rbase + i * 8;
    if (r >= it.M) continue;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const int c = cbase + j * 8;
      double* o = it.dst + (int64_t)r * it.ldd + c;
      const double v0 = it.scale * acc[i][j][0], v1 = it.scale * acc[i][j][1];
      if (vec && c + 1 < it.N) *(double2*)o = make_double2(v0, v1);
      else {
        if (c < it.N) o[0] = v0;
        if (c + 1 < it.N) o[1] = v1;
      }
    }
  }
}

template <int NI, bool LT, bool RN>
__device__ __forceinline__ void tp_consume_nj(const TpItem& it, const double* smem, uint64_t* full, uint64_t* empty, int warp, int lane, int& step) {
  switch (it.nj) {
    case 1: tp_consume<NI, 1, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    case 2: tp_consume<NI, 2, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    case 3: tp_consume<NI, 3, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    case 4: tp_consume<NI, 4, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    case 5: tp_consume<NI, 5, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    case 6: tp_consume<NI, 6, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    case 7: tp_consume<NI, 7, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    default: tp_consume<NI, 8, LT, RN>(it, smem, full, empty, warp, lane, step); break;
  }
}
template <bool LT, bool RN>
__device__ __forceinline__ void tp_consume_ni(const TpItem& it, const double* smem, uint64_t* full, uint64_t* empty, int warp, int lane, int& step) {
  switch (it.ni) {
    case 1: tp_consume_nj<1, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    case 2: tp_consume_nj<2, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    case 3: tp_consume_nj<3, LT, RN>(it, smem, full, empty, warp, lane, step); break;
    default: tp_consume_nj<4, LT, RN>(it, smem, full, empty, warp, lane, step); break;
  }
}

// warp-tile heights / widths of a ragged last tile with `rem` valid rows / columns (the instantiated sizes)
__host__ __device__ __forceinline__ int tp_ni_for(int rem) { return rem >= TP_TM ? 4 : (rem + 15) / 16; }
__host__ __device__ __forceinline__ int tp_nj_for(int rem) {
  return rem >= TP_TN ? 8 : (rem + 15) / 16;
}

// The producer's memory of the slice it is in: the items of a CTA are consecutive, so slice and task records are fetched once
// per slice, not once per item.
struct TpCache {
  int lo = -1, end = 0;     // slice index; first item beyond the slice
  TpSlice sl;
  int m, k, n, p, transA, transD, stepA, stepD;
  double coef;
  const double* alpha;
};

// What item `item` of a launch is: which slice (binary search over the slices' first items for the first item of a CTA, then
// the next slices in order), which tile, which positions.  Called by the producer thread only; the consumers get the result
// through shared memory (tp_gemm_kernel).
__device__ __forceinline__ TpItem tp_decode(const TpSlice* __restrict__ slices, int nslices, int pass, const DevTask* __restrict__ tasks,
                                            const CUtensorMap* __restrict__ maps, double* __restrict__ scratch,
                                            double* __restrict__ partial, int item, TpCache& c) {
  if (c.lo < 0 || item >= c.end) {
    if (c.lo < 0) {
      int hi = nslices - 1;
      c.lo = 0;
      while (c.lo < hi) {
        const int mid = (c.lo + hi + 1) >> 1;
        if ((pass ? slices[mid].item2 : slices[mid].item1) <= item) c.lo = mid; else hi = mid - 1;
      }
    } else {
      while (c.lo + 1 < nslices && (pass ? slices[c.lo + 1].item2 : slices[c.lo + 1].item1) <= item) ++c.lo;
    }
    c.end = c.lo + 1 < nslices ? (pass ? slices[c.lo + 1].item2 : slices[c.lo + 1].item1) : 0x7fffffff;
    c.sl = slices[c.lo];
    const DevTask* __restrict__ tk = tasks + c.sl.task;
    c.m = tk->m; c.k = tk->k; c.n = tk->n; c.p = tk->p;
    c.transA = (tk->flags & TASK_TRANS_A) != 0; c.transD = (tk->flags & TASK_TRANS_D) != 0;
    c.stepA = tk->strideA != 0; c.stepD = tk->strideD != 0;
    c.coef = tk->coef; c.alpha = tk->alpha;
  }
  const TpSlice& sl = c.sl;
  const int m = c.m, k = c.k, n = c.n, p = c.p;
  const bool transA = c.transA, transD = c.transD;
  const int stepA = c.stepA, stepD = c.stepD;
  const int local = item - (pass ? sl.item2 : sl.item1);
  TpItem it;
  int pl0;   // first position (relative to the slice) of the item
  if (pass == 0) {
    it.M = sl.order ? k : m;
    it.N = sl.order ? p : n;
    it.K = sl.order ? n : k;
  } else {
    it.M = m; it.N = p;
    it.K = sl.order ? k : n;
  }
  const int ntr = (it.M + TP_TM - 1) / TP_TM, ntc = (it.N + TP_TN - 1) / TP_TN;
  const int tile = local % (ntr * ntc), outer = local / (ntr * ntc);
  it.row0 = (tile / ntc) * TP_TM;
  it.col0 = (tile % ntc) * TP_TN;
  it.ni = tp_ni_for(it.M - it.row0);
  it.nj = tp_nj_for(it.N - it.col0);
  it.l_row = it.l_row_step = it.l_item = it.l_item_step = it.r_k = it.r_k_step = it.r_item = it.r_item_step = 0;
  const int rowsT = sl.order ? k : m;          // rows of one T_pos
  if (pass == 0) {
    pl0 = outer;
    it.npl = 1;
    it.acc_init = 0;
    const double al = c.alpha ? c.alpha[sl.pos0 + pl0] : 1.0;
    it.scale = c.coef * al;
    it.dst = scratch + ((int64_t)sl.t_row0 + (int64_t)pl0 * rowsT) * sl.ldt;
    it.ldd = sl.ldt;
    if (sl.order == 0) {   // T = Aop E
      it.mapL = maps + sl.mapA; it.lt = transA; it.l_item = stepA ? sl.pos0 + pl0 : 0;
      it.mapR = maps + sl.mapE; it.rn = 1; it.r_item = (sl.flags & TP_SLICE_E_PER_POS) ? sl.pos0 + pl0 : 0;
    } else {               // T = E Dop^T
      it.mapL = maps + sl.mapE; it.lt = 0; it.l_item = (sl.flags & TP_SLICE_E_PER_POS) ? sl.pos0 + pl0 : 0;
      it.mapR = maps + sl.mapD; it.rn = transD; it.r_item = stepD ? sl.pos0 + pl0 : 0;
    }
  } else {
    pl0 = outer * sl.chunk;
    it.npl = min(sl.chunk, sl.npos - pl0);
    it.scale = 1.0;
    it.acc_init = (sl.flags & TP_SLICE_ACCUMULATE) ? 1 : 0;
    const int64_t slab = it.acc_init ? (int64_t)m * p : ((int64_t)m * p + 1) & ~(int64_t)1;   // dense outputs / even-sized partial slabs
    it.dst = partial + sl.part_off + (int64_t)outer * slab;
    it.ldd = p;
    if (sl.order == 0) {   // partial = sum_pos T_pos Dop_pos^T
      it.mapL = maps + sl.mapT; it.lt = 0; it.l_row = sl.t_row0 + pl0 * rowsT; it.l_row_step = rowsT;
      it.mapR = maps + sl.mapD; it.rn = transD; it.r_item = stepD ? sl.pos0 + pl0 : 0; it.r_item_step = stepD;
    } else {               // partial = sum_pos Aop_pos T_pos
      it.mapL = maps + sl.mapA; it.lt = transA; it.l_item = stepA ? sl.pos0 + pl0 : 0; it.l_item_step = stepA;
      it.mapR = maps + sl.mapT; it.rn = 1; it.r_k = sl.t_row0 + pl0 * rowsT; it.r_k_step = rowsT;
    }
  }
  return it;
}

// pass = 0: T_pos of every position of the group's slices; pass = 1: the partial slabs.  Items are numbered over the group;
// CTA b works through items [b ipc, (b + 1) ipc) one after the other WITHOUT draining its pipeline in between: the producer
// thread decodes the items (tables in global memory) and hands each descriptor to the consumer warps through shared memory
// together with the item's first stage; both sides count the same stages, so the producer is already staging the next item
// while the consumers store the current one (pass 1 of small blocks: a CTA's start-up is spread over ipc items, and the
// consumers never wait for a table look-up).
__global__ void __launch_bounds__(TP_THREADS, 2)
tp_gemm_kernel(const TpSlice* __restrict__ slices, int nslices, int pass, int nitems, int ipc, const DevTask* __restrict__ tasks,
               const CUtensorMap* __restrict__ maps, double* __restrict__ scratch, double* __restrict__ partial) {
  extern __shared__ __align__(1024) double smem[];
  __shared__ __align__(8) uint64_t full[TP_NS];
  __shared__ __align__(8) uint64_t empty[TP_NS];
  __shared__ __align__(16) TpItem ring[4];        // item descriptors, producer -> consumers (TP_NS + 1 slots)
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    for (int i = 0; i < TP_NS; ++i) {
      tp_mbar_init(&full[i], 1);
      tp_mbar_init(&empty[i], TP_CONSUMERS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  const int item0 = blockIdx.x * ipc, item1 = min(nitems, item0 + ipc);
  int step = 0;
  if (warp == TP_CONSUMERS) {
    // ---- producer: one thread; per item: decode, publish the descriptor, then two boxes per stage
    if (lane != 0) return;
    TpCache cache;
    for (int item = item0; item < item1; ++item) {
      const TpItem it = tp_decode(slices, nslices, pass, tasks, maps, scratch, partial, item, cache);
      const unsigned bytes = (unsigned)(((it.lt ? TP_LBOX_M : TP_LBOX_K) + (it.rn ? TP_RBOX_N : TP_RBOX_K)) * sizeof(double));
      const int nsteps = (it.K + TP_KS - 1) / TP_KS;
      for (int pl = 0; pl < it.npl; ++pl) {
        const int lrow = it.row0 + it.l_row + pl * it.l_row_step, litem = it.l_item + pl * it.l_item_step;
        const int rk = it.r_k + pl * it.r_k_step, ritem = it.r_item + pl * it.r_item_step;
        for (int s = 0; s < nsteps; ++s, ++step) {
          const int b = step % TP_NS, round = step / TP_NS;
          if (round > 0) tp_mbar_wait(&empty[b], (round - 1) & 1);
          // The descriptor goes out with the item's first stage: written after the wait above (the consumers have released a
          // stage of item - TP_NS or later, so they are done reading slot (item - TP_NS - 1) & 3 and older) and before the
          // arrive below, whose release / the consumers' acquire on `full` make it visible to them.
          if (pl == 0 && s == 0) ring[(item - item0) & 3] = it;
          tp_mbar_expect(&full[b], bytes);
          const unsigned st = tp_smem_u32(smem + (size_t)b * TP_STAGE);
          if (it.lt) tp_tma_box(st, it.mapL, lrow, s * TP_KS, litem, &full[b]);
          else tp_tma_box(st, it.mapL, s * TP_KS, lrow, litem, &full[b]);
          if (it.rn) tp_tma_box(st + TP_LREG * 8u, it.mapR, it.col0, rk + s * TP_KS, ritem, &full[b]);
          else tp_tma_box(st + TP_LREG * 8u, it.mapR, s * TP_KS, it.col0, ritem, &full[b]);
        }
      }
    }
    return;
  }
  // ---- consumers: the descriptor of an item is valid once the item's first stage has landed
  for (int item = item0; item < item1; ++item) {
    tp_mbar_wait(&full[step % TP_NS], (step / TP_NS) & 1);
    const TpItem it = ring[(item - item0) & 3];
    if (it.lt) tp_consume_ni<true, true>(it, smem, full, empty, warp, lane, step);     // Aop read transposed: R is E or T (columns contiguous)
    else if (it.rn) tp_consume_ni<false, true>(it, smem, full, empty, warp, lane, step);
    else tp_consume_ni<false, false>(it, smem, full, empty, warp, lane, step);
  }
}

// F_s += partial slabs in index order: fixed order, one thread per element (row a5).  HBM-bound: the slabs of four
// consecutive chunks are fetched before they are added (the additions stay in index order).
__global__ void __launch_bounds__(256)
tp_reduce_kernel(const TpReduce* __restrict__ red, const double* __restrict__ partial, double* __restrict__ out) {
  const TpReduce r = red[blockIdx.y];
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < r.size; i += (int64_t)gridDim.x * blockDim.x) {
    double s = out[r.f_off + i];
    const double* __restrict__ q = partial + r.part_off + i;
    int g = 0;
    for (; g + 4 <= r.nslab; g += 4) {
      const double a = q[(int64_t)g * r.slab], b = q[(int64_t)(g + 1) * r.slab], c = q[(int64_t)(g + 2) * r.slab], d = q[(int64_t)(g + 3) * r.slab];
      s += a; s += b; s += c; s += d;
    }
    for (; g < r.nslab; ++g) s += q[(int64_t)g * r.slab];
    out[r.f_off + i] = s;
  }
}

}  // namespace

int tp_tile_rows_executed(int M) {   // rows the row tiles of an M-row output multiply (host: executed flops)
  const int full = M / TP_TM, rem = M % TP_TM;
  return full * TP_TM + (rem ? 16 * tp_ni_for(rem) : 0);
}
int tp_tile_cols_executed(int N) {
  const int full = N / TP_TN, rem = N % TP_TN;
  return full * TP_TN + (rem ? 16 * tp_nj_for(rem) : 0);
}

static su2_status tp_set_attr() {
  static bool attr_done[64] = {};
  int dev = 0;
  cudaGetDevice(&dev);
  if (!attr_done[dev & 63]) {
    cudaError_t e = cudaFuncSetAttribute(tp_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TP_SMEM);
    if (e != cudaSuccess) { set_cuda_error("cudaFuncSetAttribute(tp_gemm_kernel)", (int)e); return SU2_ERR_CUDA; }
    attr_done[dev & 63] = true;
  }
  return SU2_OK;
}

su2_status launch_tp_gemm(const TpSlice* slices, int nslices, int pass, int nitems, int ipc, const DevTask* tasks, const void* maps,
                          double* scratch, double* partial, void* stream_v) {
  su2_status st = tp_set_attr();
  if (st != SU2_OK) return st;
  if (nitems <= 0) return SU2_OK;
  ipc = std::max(1, ipc);
  tp_gemm_kernel<<<(nitems + ipc - 1) / ipc, TP_THREADS, TP_SMEM, (cudaStream_t)stream_v>>>(slices, nslices, pass, nitems, ipc, tasks,
                                                                                           (const CUtensorMap*)maps, scratch, partial);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_cuda_error("tp_gemm_kernel launch", (int)e); return SU2_ERR_CUDA; }
  count_launch();
  return SU2_OK;
}

su2_status launch_heff_two_pass(const su2_plan* plan, double* out, double* tp_partial, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  if (plan->h_tp_groups.empty()) return SU2_OK;
  static bool attr_done[64] = {};
  int dev = 0;
  cudaGetDevice(&dev);
  if (!attr_done[dev & 63]) {
    cudaError_t e = cudaFuncSetAttribute(tp_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TP_SMEM);
    if (e != cudaSuccess) { set_cuda_error("cudaFuncSetAttribute(tp_gemm_kernel)", (int)e); return SU2_ERR_CUDA; }
    attr_done[dev & 63] = true;
  }
  for (const TpGroup& g : plan->h_tp_groups) {
    const int ns = g.slice1 - g.slice0;
    tp_gemm_kernel<<<(g.items1 + g.ipc1 - 1) / g.ipc1, TP_THREADS, TP_SMEM, stream>>>(plan->d_tp_slices + g.slice0, ns, 0, g.items1, g.ipc1, plan->d_tasks,
                                                                                     (const CUtensorMap*)plan->d_maps, plan->d_tp_scratch, tp_partial);
    tp_gemm_kernel<<<g.items2, TP_THREADS, TP_SMEM, stream>>>(plan->d_tp_slices + g.slice0, ns, 1, g.items2, 1, plan->d_tasks,
                                                             (const CUtensorMap*)plan->d_maps, plan->d_tp_scratch, tp_partial);
    dim3 grid(296, (unsigned)(g.red1 - g.red0));   // few records per group (often one output sector): many CTAs per record
    tp_reduce_kernel<<<grid, 256, 0, stream>>>(plan->d_tp_reduce + g.red0, tp_partial, out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_cuda_error("two-pass launch", (int)e); return SU2_ERR_CUDA; }
    count_launch(3);
  }
  return SU2_OK;
}

}  // namespace su2
