// sm_100a fused GEMM-pair kernel of the hot path:
//
//   F_tile (TM x TP, registers) += sum_{task, pos} (coef alpha_pos) * (A_pos[rows,:] E) D_pos[cols,:]^T
//
// the paper's two SBGEMM steps fused per task: the intermediate T = A_pos E
// never leaves the SM (accumulated in registers, parked in shared memory as the A operand of the
// second product), and the sum over positions is the K loop of the second product (the paper's
// stripe trick).
//
// Arithmetic: FP64 tensor instructions mma.sync.aligned.m8n8k4.f64 (SASS DMMA.8x8x4) -- the only
// FP64 matrix instruction sm_100a exposes (tcgen05 has no f64 kind); measured at 37.1 TFLOP/s =
// 99.8 % of 148 SM x 64 FMA/clk x 1.965 GHz, against 33.8 TFLOP/s for a DFMA loop
// (profiles/r01_fp64_peak_probe.txt).
//
// Structure: persistent CTAs (one per SM, 8 warps) pull work items (segment x output tile) from an
// atomic queue in the plan's longest-first order.  Inside an item every (task, position, T-chunk)
// is a run of pipeline *steps*: first-product steps (A tile + E tile, KS deep) followed by
// second-product steps (D tile, KS deep).  Steps are described by small descriptors that one
// thread generates ahead of time into a shared-memory ring, so the control state costs no
// registers; operand tiles are staged by 8-byte cp.async with zero fill (ragged block sizes and
// odd leading dimensions need no special cases) NSTAGE-1 steps ahead of the math.
#include <cuda_runtime.h>

#include <algorithm>

#include "su2_internal.h"
#include "tile_config.h"

namespace su2 {

namespace {

enum : int { STEP_END = 1, STEP_G2 = 2, STEP_TRANS = 4, STEP_FIRST = 8, STEP_LAST = 16 };

struct StepDesc {
  const double* src0;   // first product: A tile origin;  second product: D tile origin
  const double* src1;   // first product: E tile origin
  double scale;         // coef * alpha_pos, applied when the last first-product step parks T
  int ld0, ld1;         // global leading dimensions
  int cval0;            // valid extent of tile 0 along c (rows of A / columns of F)
  int cval1;            // valid columns of the E tile (= width of the T chunk)
  int jval;             // valid extent along k (<= KS)
  int s;                // step index inside its phase
  int flags;
  int pad;
};

struct GenState {       // iterator over the steps of one work item (lives in shared memory)
  const double *A, *D, *E, *alpha;
  double coef, scale;
  int m, k, n, p, strideA, strideD, tflags;
  int u, u_end, pos, pos_end, chunk, nchunks, ncw_full, n0, ncw, phase, s, nsteps1, nsteps2, done;
  int row0, col0, rows_valid, cols_valid, nc_max;
};

constexpr int RING = NSTAGE + 1;

__device__ __forceinline__ void gen_set_chunk(GenState& st) {
  st.n0 = st.chunk * st.ncw_full;
  st.ncw = min(st.ncw_full, st.n - st.n0);
  st.nsteps2 = (st.ncw + KS - 1) / KS;
  st.phase = 0;
  st.s = 0;
}
__device__ __forceinline__ void gen_set_pos(GenState& st) {
  st.scale = st.coef * (st.alpha ? st.alpha[st.pos] : 1.0);
  st.chunk = 0;
  gen_set_chunk(st);
}
__device__ __forceinline__ void gen_load_unit(GenState& st, const DevUnit* __restrict__ units,
                                              const DevTask* __restrict__ tasks, const double* __restrict__ psi) {
  const DevUnit un = units[st.u];
  const DevTask& t = tasks[un.task];
  st.A = t.A; st.D = t.D; st.alpha = t.alpha; st.coef = t.coef; st.E = psi + t.e_off;
  st.m = t.m; st.k = t.k; st.n = t.n; st.p = t.p;
  st.strideA = t.strideA; st.strideD = t.strideD; st.tflags = (int)t.flags;
  st.pos = un.pos0; st.pos_end = un.pos1;
  st.nsteps1 = (t.k + KS - 1) / KS;
  chunking(t.n, st.nc_max, st.nchunks, st.ncw_full);
  gen_set_pos(st);
}

// Emit the descriptor of the current step and advance the iterator (one thread).
__device__ void gen_step(GenState& st, StepDesc& d, const DevUnit* __restrict__ units,
                         const DevTask* __restrict__ tasks, const double* __restrict__ psi) {
  if (st.done) {
    d.flags = STEP_END;
    return;
  }
  if (st.phase == 0) {
    const int k0 = st.s * KS;
    const bool tr = st.tflags & TASK_TRANS_A;
    d.src0 = st.A + (int64_t)st.pos * st.strideA +
             (tr ? (int64_t)k0 * st.m + st.row0 : (int64_t)st.row0 * st.k + k0);
    d.ld0 = tr ? st.m : st.k;
    d.src1 = st.E + (int64_t)k0 * st.n + st.n0;
    d.ld1 = st.n;
    d.cval0 = st.rows_valid;
    d.cval1 = st.ncw;
    d.jval = min(KS, st.k - k0);
    d.s = st.s;
    d.scale = st.scale;
    d.flags = (tr ? STEP_TRANS : 0) | (st.s == 0 ? STEP_FIRST : 0) | (st.s == st.nsteps1 - 1 ? STEP_LAST : 0);
  } else {
    const int j0 = st.n0 + st.s * KS;
    const bool tr = st.tflags & TASK_TRANS_D;
    d.src0 = st.D + (int64_t)st.pos * st.strideD +
             (tr ? (int64_t)j0 * st.p + st.col0 : (int64_t)st.col0 * st.n + j0);
    d.ld0 = tr ? st.p : st.n;
    d.cval0 = st.cols_valid;
    d.jval = min(KS, st.ncw - st.s * KS);
    d.s = st.s;
    d.flags = STEP_G2 | (tr ? STEP_TRANS : 0);
  }
  ++st.s;
  if (st.phase == 0) {
    if (st.s == st.nsteps1) { st.phase = 1; st.s = 0; }
  } else if (st.s == st.nsteps2) {
    if (++st.chunk < st.nchunks) gen_set_chunk(st);
    else if (++st.pos < st.pos_end) gen_set_pos(st);
    else if (++st.u < st.u_end) gen_load_unit(st, units, tasks, psi);
    else st.done = 1;
  }
}

// ---- cp.async staging (8-byte elements, zero fill when !valid) ---------------------------
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* src, bool valid) {
  const unsigned dst = (unsigned)__cvta_generic_to_shared(smem_dst);
  const int sz = valid ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// Both copies land in the same shared-memory layout, [j/4][j%4][c] with row stride CT+4 doubles
// (k-major k4 sub-tiles; CT+4 = 4 mod 8 makes the DMMA fragment loads conflict-free), so the math
// code does not depend on how the operator block is stored.
// Source stored c-major, element (c, j) = src[c*ld + j]: 8 consecutive lanes read one 64-byte run.
template <int CT>
__device__ __forceinline__ void copy_cmajor(double* dst, const double* __restrict__ src, int ld, int cval, int jval) {
  const int cpad = (cval + 7) & ~7;
  const int jpad = jval > 4 ? 8 : 4;
  const int j = threadIdx.x & 7;
  if (j >= jpad) return;
  double* d = dst + (j >> 2) * (4 * (CT + 4)) + (j & 3) * (CT + 4);
  const bool jok = j < jval;
  for (int c = threadIdx.x >> 3; c < cpad; c += NTHREADS / 8) {
    const bool ok = jok && c < cval;
    cp_async8(d + c, ok ? src + (int64_t)c * ld + j : src, ok);
  }
}
// Source stored k-major, element (c, j) = src[j*ld + c]: a warp reads one 256-byte run.
template <int CT>
__device__ __forceinline__ void copy_kmajor(double* dst, const double* __restrict__ src, int ld, int cval, int jval) {
  const int cpad = (cval + 7) & ~7;
  const int jpad = jval > 4 ? 8 : 4;
  for (int j = 0; j < jpad; ++j) {
    double* d = dst + (j >> 2) * (4 * (CT + 4)) + (j & 3) * (CT + 4);
    const double* s = src + (int64_t)j * ld;
    const bool jok = j < jval;
    for (int c = threadIdx.x; c < cpad; c += NTHREADS) {
      const bool ok = jok && c < cval;
      cp_async8(d + c, ok ? s + c : src, ok);
    }
  }
}

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}

// One pipeline stage (nsub k4 sub-steps) of a warp-level product: c[ii][j] += A_frag[ii] B_frag[j]
// for 4 m8-tiles (the first mt active) and NT n8-tiles.  a / b point at this lane's element of the
// first fragment; A_I / A_SUB / B_SUB are the compile-time strides between m8-tiles / k4 sub-steps
// (n8-tiles are 8 doubles apart).
template <int NT, int NACC, int A_I, int A_SUB, int B_SUB>
__device__ __forceinline__ void mma_stage(double (&c)[4][NACC][2], const double* __restrict__ a,
                                          const double* __restrict__ b, int nsub, int mt) {
#pragma unroll
  for (int sub = 0; sub < 2; ++sub) {
    if (sub < nsub) {
      double af[4], bf[NT];
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) af[ii] = a[sub * A_SUB + ii * A_I];
#pragma unroll
      for (int j = 0; j < NT; ++j) bf[j] = b[sub * B_SUB + j * 8];
      if (mt == 4) {
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) dmma(c[ii][j], af[ii], bf[j]);
      } else {
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
          for (int ii = 0; ii < 3; ++ii)
            if (ii < mt) dmma(c[ii][j], af[ii], bf[j]);
      }
    }
  }
}

template <int WR>
__device__ __forceinline__ void issue_loads(const StepDesc& d, double* stage) {
  using C = TileCfg<WR>;
  const int flags = d.flags;
  if (flags & STEP_END) return;
  if (!(flags & STEP_G2)) {
    if (flags & STEP_TRANS) copy_kmajor<C::TM>(stage, d.src0, d.ld0, d.cval0, d.jval);
    else copy_cmajor<C::TM>(stage, d.src0, d.ld0, d.cval0, d.jval);
    copy_kmajor<C::NC>(stage + C::A_SZ, d.src1, d.ld1, d.cval1, d.jval);
  } else {
    if (flags & STEP_TRANS) copy_kmajor<C::TP>(stage, d.src0, d.ld0, d.cval0, d.jval);
    else copy_cmajor<C::TP>(stage, d.src0, d.ld0, d.cval0, d.jval);
  }
}

// One work item: TM x TP tile of one output sector, one segment of its (task, position) list.
template <int WR>
__device__ void run_item(const DevWork& wk, const DevUnit* __restrict__ units, const DevTask* __restrict__ tasks,
                         const double* __restrict__ psi, double* __restrict__ dst, double* smem, GenState& st,
                         StepDesc* ring) {
  using C = TileCfg<WR>;
  constexpr int WC = C::WC, TM = C::TM, TP = C::TP, NC = C::NC, LDT = C::LDT, LDE = NC + 4;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
  const int wr = warp / WC, wc = warp % WC;
  double* Ts = smem;
  double* stages = smem + TM * LDT;

  const int rows_valid = min(TM, wk.m - wk.row0);
  const int cols_valid = min(TP, wk.p - wk.col0);
  const int mt = max(0, min(4, (rows_valid - wr * 32 + 7) >> 3));          // active m8-tiles of this warp
  const int ntiles2 = (cols_valid + 7) >> 3;
  const int ntw2 = (ntiles2 + WC - 1) / WC;
  const int ctile0 = wc * ntw2;
  const int nt2 = max(0, min(ntw2, ntiles2 - ctile0));                     // active n8-tiles (second product)

  if (tid == 0) {
    st.u = wk.unit0; st.u_end = wk.unit1; st.done = 0;
    st.row0 = wk.row0; st.col0 = wk.col0; st.rows_valid = rows_valid; st.cols_valid = cols_valid; st.nc_max = NC;
    if (st.u < st.u_end) gen_load_unit(st, units, tasks, psi);
    else st.done = 1;
    for (int i = 0; i < NSTAGE; ++i) gen_step(st, ring[i], units, tasks, psi);
  }
  __syncthreads();
#pragma unroll 1
  for (int L = 0; L < NSTAGE - 1; ++L) {
    issue_loads<WR>(ring[L], stages + L * C::STAGE);
    cp_async_commit();
  }

  double acc[4][NT2][2];
  double tacc[4][NT1][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < NT2; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < NT1; ++j) tacc[i][j][0] = tacc[i][j][1] = 0.0;

  int slot = 0;          // ring slot of step i
  int buf = 0;           // stage buffer of step i
#pragma unroll 1
  for (int i = 0;; ++i) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();
    const StepDesc& d = ring[slot];
    const int flags = d.flags;
    if (flags & STEP_END) break;
    {   // stage the operands of step i + NSTAGE - 1 into the buffer that step i - 1 has just released
      int lslot = slot + NSTAGE - 1; if (lslot >= RING) lslot -= RING;
      int lbuf = buf + NSTAGE - 1;  if (lbuf >= NSTAGE) lbuf -= NSTAGE;
      issue_loads<WR>(ring[lslot], stages + lbuf * C::STAGE);
      cp_async_commit();
      if (tid == ((i & 7) << 5)) {       // descriptor of step i + NSTAGE, written into the slot of step i - 1
        int gslot = lslot + 1; if (gslot >= RING) gslot -= RING;
        gen_step(st, ring[gslot], units, tasks, psi);
      }
    }
    const double* stage = stages + buf * C::STAGE;
    const int nsub = d.jval > 4 ? 2 : 1;
    if (!(flags & STEP_G2)) {
      // ---- first product: tacc (32 x 8 NT1 per warp) += A_tile E_tile --------------------------
      const int ntiles1 = (d.cval1 + 7) >> 3;
      const int nt1w = (ntiles1 + WC - 1) / WC;
      const int tile0 = wc * nt1w;
      const int nt1 = max(0, min(nt1w, ntiles1 - tile0));
      const double* a = stage + t * (TM + 4) + wr * 32 + g;
      const double* b = stage + C::A_SZ + t * LDE + tile0 * 8 + g;
      if (flags & STEP_FIRST) {
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int j = 0; j < NT1; ++j) tacc[ii][j][0] = tacc[ii][j][1] = 0.0;
      }
      if (mt > 0) {
        switch (nt1) {
          case 1: mma_stage<1, NT1, 8, 4 * (TM + 4), 4 * LDE>(tacc, a, b, nsub, mt); break;
          case 2: mma_stage<2, NT1, 8, 4 * (TM + 4), 4 * LDE>(tacc, a, b, nsub, mt); break;
          case 3: mma_stage<3, NT1, 8, 4 * (TM + 4), 4 * LDE>(tacc, a, b, nsub, mt); break;
          case 4: mma_stage<4, NT1, 8, 4 * (TM + 4), 4 * LDE>(tacc, a, b, nsub, mt); break;
          default: break;
        }
      }
      if (flags & STEP_LAST) {
        const double sc = d.scale;
        double* trow = Ts + (wr * 32 + g) * LDT + tile0 * 8 + 2 * t;
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int j = 0; j < NT1; ++j)
            if (ii < mt && j < nt1)
              *reinterpret_cast<double2*>(trow + ii * 8 * LDT + j * 8) = make_double2(sc * tacc[ii][j][0], sc * tacc[ii][j][1]);
      }
    } else {
      // ---- second product: acc (32 x 8 NT2 per warp) += T_chunk[:, step] D_tile^T ---------------
      const double* a = Ts + (wr * 32 + g) * LDT + d.s * KS + t;
      const double* b = stage + t * (TP + 4) + ctile0 * 8 + g;
      if (mt > 0) {
        switch (nt2) {
          case 1: mma_stage<1, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          case 2: mma_stage<2, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          case 3: mma_stage<3, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          case 4: mma_stage<4, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          case 5: mma_stage<5, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          case 6: mma_stage<6, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          case 7: mma_stage<7, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          case 8: mma_stage<8, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          case 9: mma_stage<9, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, a, b, nsub, mt); break;
          default: break;
        }
      }
    }
    if (++slot == RING) slot = 0;
    if (++buf == NSTAGE) buf = 0;
  }
  cp_async_wait<0>();

  // ---- epilogue: the tile leaves the registers once per work item -----------------------------
#pragma unroll
  for (int ii = 0; ii < 4; ++ii)
#pragma unroll
    for (int j = 0; j < NT2; ++j)
      if (ii < mt && j < nt2) {
        const int r = wk.row0 + wr * 32 + ii * 8 + g;
        const int q = wk.col0 + (ctile0 + j) * 8 + 2 * t;
        if (r < wk.m) {
          double* o = dst + (int64_t)r * wk.p + q;
          if (q < wk.p) o[0] = acc[ii][j][0];
          if (q + 1 < wk.p) o[1] = acc[ii][j][1];
        }
      }
}

__global__ void __launch_bounds__(NTHREADS, 1)
heff_dmma_kernel(const DevWork* __restrict__ work, int nwork, const DevUnit* __restrict__ units,
                 const DevTask* __restrict__ tasks, const double* __restrict__ psi, double* __restrict__ out,
                 double* __restrict__ partial, int* __restrict__ counter) {
  extern __shared__ __align__(16) double smem[];
  __shared__ GenState st;
  __shared__ StepDesc ring[RING];
  __shared__ int s_w;
  for (;;) {
    __syncthreads();                       // previous item fully retired (smem, ring, s_w)
    if (threadIdx.x == 0) s_w = atomicAdd(counter, 1);
    __syncthreads();
    const int w = s_w;
    if (w >= nwork) break;
    const DevWork wk = work[w];
    double* dst = (wk.to_partial ? partial : out) + wk.dst_off;
    if (wk.wr == 1) run_item<1>(wk, units, tasks, psi, dst, smem, st, ring);
    else if (wk.wr == 2) run_item<2>(wk, units, tasks, psi, dst, smem, st, ring);
    else run_item<4>(wk, units, tasks, psi, dst, smem, st, ring);
  }
}

}  // namespace

su2_status launch_heff_dmma(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  const int nwork = (int)plan->h_work.size();
  if (nwork == 0) return SU2_OK;
  static bool attr_set = false;
  const size_t smem_bytes = (size_t)SMEM_DOUBLES_MAX * sizeof(double);
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(heff_dmma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) { set_cuda_error("cudaFuncSetAttribute(heff_dmma_kernel)", (int)e); return SU2_ERR_CUDA; }
    attr_set = true;
  }
  const int grid = std::min(nwork, plan->num_sms);
  heff_dmma_kernel<<<grid, NTHREADS, smem_bytes, stream>>>(plan->d_work, nwork, plan->d_units, plan->d_tasks, psi, out,
                                                           partial, plan->d_counter);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_cuda_error("heff_dmma_kernel launch", (int)e); return SU2_ERR_CUDA; }
  count_launch();
  return SU2_OK;
}

}  // namespace su2
