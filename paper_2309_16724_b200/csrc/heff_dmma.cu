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
// Structure: persistent CTAs (one per SM) pull work items (segment x output tile) from an atomic
// queue in the plan's longest-first order.  Inside an item every (task, position, T-chunk) is a run
// of pipeline *steps*: first-product steps (A tile + E tile, KS deep) followed by second-product
// steps (D tile, KS deep).  The CTA is warp-specialised:
//   * warps 0-3 (one warpgroup, 40 registers after setmaxnreg.dec) are PRODUCERS.  Producer warp w
//     owns stage buffer w: it walks the item's step sequence with an iterator kept in shared
//     memory, writes the step descriptor, and stages the operand tiles with 8-byte cp.async + zero
//     fill (ragged block sizes and odd leading dimensions need no special cases); completion is
//     signalled on an mbarrier (cp.async.mbarrier.arrive.noinc).
//   * warps 4-11 (two warpgroups, 232 registers after setmaxnreg.inc) are CONSUMERS: they wait on
//     the stage's "full" mbarrier, issue only LDS + DMMA, and release the stage on its "empty"
//     mbarrier.  No CTA-wide barrier exists inside an item; the T hand-over between the two
//     products uses a named barrier of the 256 consumer threads.
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

struct GenState {       // iterator over the steps of one work item (one per producer warp, in shared memory)
  const double *A, *D, *E, *alpha;
  double coef, scale;
  int m, k, n, p, strideA, strideD, tflags;
  int u, u_end, pos, pos_end, chunk, nchunks, ncw_full, n0, ncw, phase, s, nsteps1, nsteps2, done;
  int row0, col0, rows_valid, cols_valid, nc_max;
};

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

// Move the iterator to the next step.
__device__ __forceinline__ void gen_advance(GenState& st, const DevUnit* __restrict__ units,
                                            const DevTask* __restrict__ tasks, const double* __restrict__ psi) {
  if (st.done) return;
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

// Descriptor of the current step.
__device__ __forceinline__ void gen_fill(const GenState& st, StepDesc& d) {
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
}

// ---- PTX helpers -------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, int parity) {
  unsigned ok;
  asm volatile(
      "{\n.reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, int parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
// arrive on `bar` once all cp.async issued so far by this thread have landed (count pre-charged at init)
__device__ __forceinline__ void cp_async_mbar_arrive(uint64_t* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, 256;\n" ::: "memory"); }
__device__ __forceinline__ void cta_bar() { asm volatile("bar.sync 0, 384;\n" ::: "memory"); }
static_assert(NTHREADS == 384 && NWARPS * 32 == 256, "barrier thread counts are spelled out in the PTX above");

// ---- staging: one producer WARP copies a whole tile ---------------------------------------------
// Every tile lands in the same shared-memory layout, [j/4][j%4][c] with row stride CT+4 doubles
// (k-major k4 sub-tiles; CT+4 = 4 mod 8 makes the DMMA fragment loads conflict-free), so the math
// code does not depend on how the operator block is stored.
// The copy loops are written with running addresses (one LDGSTS + two adds per element): a single
// producer warp has to issue a whole tile, so its instruction count is what bounds the pipeline.
__device__ __forceinline__ void cp_async8_raw(unsigned dst, const void* src, int sz) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
// Source stored c-major, element (c, j) = src[c*ld + j]: 8 consecutive lanes read one 64-byte run.
template <int CT>
__device__ __forceinline__ void copy_cmajor(double* dst, const double* __restrict__ src, int ld, int cval, int jval, int lane) {
  const int j = lane & 7, r = lane >> 3;
  if (j >= (jval > 4 ? 8 : 4)) return;
  unsigned d = smem_u32(dst + (j >> 2) * (4 * (CT + 4)) + (j & 3) * (CT + 4) + r);
  const char* s = reinterpret_cast<const char*>(src + (int64_t)r * ld + j);
  const int64_t sstep = (int64_t)ld * 32;            // four rows further
  const int szj = j < jval ? 8 : 0;
  const int ntot = ((cval + 7) & ~7) >> 2;           // iterations up to the padded extent
  const int nfull = min(ntot, max(0, (cval - r + 3) >> 2));
  int i = 0;
#pragma unroll 4
  for (; i < nfull; ++i) {
    cp_async8_raw(d, s, szj);
    d += 32;
    s += sstep;
  }
  for (; i < ntot; ++i) {                            // rows beyond the block: zero fill
    cp_async8_raw(d, src, 0);
    d += 32;
  }
}
// Source stored k-major, element (c, j) = src[j*ld + c]: a warp reads one 256-byte run.
template <int CT>
__device__ __forceinline__ void copy_kmajor(double* dst, const double* __restrict__ src, int ld, int cval, int jval, int lane) {
  const int cpad = (cval + 7) & ~7;
  const int jpad = jval > 4 ? 8 : 4;
#pragma unroll 1
  for (int j = 0; j < jpad; ++j) {
    unsigned d = smem_u32(dst + (j >> 2) * (4 * (CT + 4)) + (j & 3) * (CT + 4) + lane);
    const char* s = reinterpret_cast<const char*>(src + (int64_t)j * ld + lane);
    const int szj = j < jval ? 8 : 0;
    int c = lane;
#pragma unroll 4
    for (; c < cval; c += 32) {
      cp_async8_raw(d, s, szj);
      d += 256;
      s += 256;
    }
    if (c < cpad) cp_async8_raw(d, src, 0);          // at most one padded element per lane
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

// ---- producer warp w: owns stage buffer w and the item's steps  l  with (base + l) % NSTAGE == w --------
// Descriptors are double-buffered per stage (ring[fill parity][w]): the descriptor of the next fill
// is generated while the current fill is in flight, off the critical path of the buffer hand-over.
template <int WR>
__device__ __forceinline__ void producer_item(const DevWork& wk, const DevUnit* __restrict__ units,
                                              const DevTask* __restrict__ tasks, const double* __restrict__ psi,
                                              double* smem, GenState& st, StepDesc (*ring)[NSTAGE], uint64_t* full,
                                              uint64_t* empty, int w, int lane, int first, unsigned& nfill) {
  using C = TileCfg<WR>;
  double* stage = smem + C::TM * C::LDT + w * C::STAGE;
  if (lane == 0) {
    st.u = wk.unit0; st.u_end = wk.unit1; st.done = 0;
    st.row0 = wk.row0; st.col0 = wk.col0;
    st.rows_valid = min(C::TM, wk.m - wk.row0);
    st.cols_valid = min(C::TP, wk.p - wk.col0);
    st.nc_max = C::NC;
    if (st.u < st.u_end) gen_load_unit(st, units, tasks, psi);
    else st.done = 1;
    for (int i = 0; i < first; ++i) gen_advance(st, units, tasks, psi);
    gen_fill(st, ring[nfill & 1u][w]);
#pragma unroll 1
    for (int i = 0; i < NSTAGE; ++i) gen_advance(st, units, tasks, psi);
  }
#pragma unroll 1
  for (;;) {
    __syncwarp();                                       // descriptor of this fill is visible to the warp
    const StepDesc& desc = ring[nfill & 1u][w];
    mbar_wait(&empty[w], (int)((nfill & 1u) ^ 1u));     // consumers have released the previous fill of this buffer
    const int flags = desc.flags;
    if (!(flags & STEP_END)) {
      const double* src0 = desc.src0;
      const int ld0 = desc.ld0, cval0 = desc.cval0, jval = desc.jval;
      if (!(flags & STEP_G2)) {
        if (flags & STEP_TRANS) copy_kmajor<C::TM>(stage, src0, ld0, cval0, jval, lane);
        else copy_cmajor<C::TM>(stage, src0, ld0, cval0, jval, lane);
        copy_kmajor<C::NC>(stage + C::A_SZ, desc.src1, desc.ld1, desc.cval1, jval, lane);
      } else {
        if (flags & STEP_TRANS) copy_kmajor<C::TP>(stage, src0, ld0, cval0, jval, lane);
        else copy_cmajor<C::TP>(stage, src0, ld0, cval0, jval, lane);
      }
    }
    cp_async_mbar_arrive(&full[w]);          // 32 deferred arrivals: this lane's copies have landed
    __syncwarp();
    if (lane == 0) mbar_arrive(&full[w]);    // +1 (release): the descriptor is visible
    ++nfill;
    if (flags & STEP_END) break;
    if (lane == 0) {                         // next descriptor, while this fill is in flight
      gen_fill(st, ring[nfill & 1u][w]);
#pragma unroll 1
      for (int i = 0; i < NSTAGE; ++i) gen_advance(st, units, tasks, psi);
    }
  }
}

// ---- consumer warp cw = (wr, wc): LDS + DMMA only -------------------------------------------------------
template <int WR>
__device__ __forceinline__ void consumer_item(const DevWork& wk, double* __restrict__ dst, double* smem,
                                              const StepDesc (*ring)[NSTAGE], uint64_t* full, uint64_t* empty, int cw, int lane,
                                              unsigned& ci) {
  using C = TileCfg<WR>;
  constexpr int WC = C::WC, TM = C::TM, TP = C::TP, NC = C::NC, LDT = C::LDT, LDE = NC + 4;
  const int g = lane >> 2, t = lane & 3;
  const int wr = cw / WC, wc = cw % WC;
  double* Ts = smem;
  const double* stages = smem + TM * LDT;

  const int rows_valid = min(TM, wk.m - wk.row0);
  const int cols_valid = min(TP, wk.p - wk.col0);
  const int mt = max(0, min(4, (rows_valid - wr * 32 + 7) >> 3));          // active m8-tiles of this warp
  const int ntiles2 = (cols_valid + 7) >> 3;
  const int ntw2 = (ntiles2 + WC - 1) / WC;
  const int ctile0 = wc * ntw2;
  const int nt2 = max(0, min(ntw2, ntiles2 - ctile0));                     // active n8-tiles (second product)

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

  int ends = 0;
#pragma unroll 1
  for (;;) {
    const int buf = (int)(ci & (NSTAGE - 1));
    const unsigned par = (ci >> 2) & 1u;
    mbar_wait(&full[buf], (int)par);
    ++ci;
    const StepDesc& d = ring[par][buf];
    const int flags = d.flags;
    if (flags & STEP_END) {
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[buf]);
      if (++ends == NSTAGE) break;
      continue;
    }
    const double* stage = stages + buf * C::STAGE;
    const int nsub = d.jval > 4 ? 2 : 1;
    if (!(flags & STEP_G2)) {
      // ---- first product: tacc (32 x 8 NT1 per warp) += A_tile E_tile --------------------------
      const int ntiles1 = (d.cval1 + 7) >> 3;
      const int nt1w = (ntiles1 + WC - 1) / WC;
      const int tile0 = wc * nt1w;
      const int nt1 = max(0, min(nt1w, ntiles1 - tile0));
      const double sc = d.scale;
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
          default: break;
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[buf]);       // stage (and its descriptor) released
      if (flags & STEP_LAST) {
        consumer_bar();                              // every warp is done reading the previous T chunk
        double* trow = Ts + (wr * 32 + g) * LDT + tile0 * 8 + 2 * t;
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int j = 0; j < NT1; ++j)
            if (ii < mt && j < nt1)
              *reinterpret_cast<double2*>(trow + ii * 8 * LDT + j * 8) = make_double2(sc * tacc[ii][j][0], sc * tacc[ii][j][1]);
        consumer_bar();                              // the new T chunk is visible to every warp
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
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[buf]);
    }
  }

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
  __shared__ GenState gs[NPRODUCERS];
  __shared__ StepDesc ring[2][NSTAGE];
  __shared__ __align__(8) uint64_t full[NSTAGE];
  __shared__ __align__(8) uint64_t empty[NSTAGE];
  __shared__ int s_w, s_base;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    for (int i = 0; i < NSTAGE; ++i) {
      mbar_init(&full[i], 32 + 1);      // 32 deferred cp.async arrivals + the descriptor writer
      mbar_init(&empty[i], NWARPS);     // one arrival per consumer warp
    }
    s_base = 0;
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  if (warp < NPRODUCERS) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n");
    unsigned nfill = 0;                  // fills of this warp's stage buffer so far (mbarrier phase)
#pragma unroll 1
    for (;;) {
      cta_bar();                         // previous item retired; s_base published
      if (tid == 0) s_w = atomicAdd(counter, 1);
      cta_bar();
      const int w = s_w;
      if (w >= nwork) break;
      const DevWork wk = work[w];
      const int first = (warp - s_base) & (NSTAGE - 1);
      if (wk.wr == 1) producer_item<1>(wk, units, tasks, psi, smem, gs[warp], ring, full, empty, warp, lane, first, nfill);
      else if (wk.wr == 2) producer_item<2>(wk, units, tasks, psi, smem, gs[warp], ring, full, empty, warp, lane, first, nfill);
      else producer_item<4>(wk, units, tasks, psi, smem, gs[warp], ring, full, empty, warp, lane, first, nfill);
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;\n");
    unsigned ci = 0;                     // steps consumed so far: stage buffer = ci % NSTAGE, phase = ci / NSTAGE
    const int cw = warp - NPRODUCERS;
#pragma unroll 1
    for (;;) {
      cta_bar();
      cta_bar();
      const int w = s_w;
      if (w >= nwork) break;
      const DevWork wk = work[w];
      double* dst = (wk.to_partial ? partial : out) + wk.dst_off;
      if (wk.wr == 1) consumer_item<1>(wk, dst, smem, ring, full, empty, cw, lane, ci);
      else if (wk.wr == 2) consumer_item<2>(wk, dst, smem, ring, full, empty, cw, lane, ci);
      else consumer_item<4>(wk, dst, smem, ring, full, empty, cw, lane, ci);
      if (tid == NPRODUCERS * 32) s_base = (int)(ci & (NSTAGE - 1));
    }
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
