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
// queue in the plan's longest-first order.  Inside an item every (task, position, T-chunk) is a pair
// of *phases*: the first product (stages of an A tile + an E tile, KS1 deep) and the second product
// (stages of a D tile, KS2 deep).  The CTA is warp-specialised:
//   * warps 0-3 (one warpgroup, 56 registers after setmaxnreg.dec) are PRODUCERS.  Every producer warp
//     walks every stage and copies a quarter of its tiles with cp.async + zero fill (ragged block sizes
//     and odd leading dimensions need no special cases): 16-byte copies for sources read along their
//     contiguous direction (E tiles, blocks read transposed -- which includes the plan's transposed
//     copies of the right-block families), 8-byte copies for the small row-major A tiles.  Completion is
//     signalled on the stage's "full" mbarrier (cp.async.mbarrier.arrive.noinc).  Lane 0 of warp 0 also
//     runs the phase iterator (state in shared memory) one phase ahead into a ring of phase descriptors.
//   * warps 4-11 (two warpgroups, 224 registers after setmaxnreg.inc) are CONSUMERS: they wait on
//     the stage's "full" mbarrier, issue only LDS + DMMA, and release the stage on its "empty"
//     mbarrier.  No CTA-wide barrier exists inside an item; the T hand-over between the two
//     products uses a named barrier of the 256 consumer threads.
#include <cuda_runtime.h>

#include <algorithm>

#include "su2_internal.h"
#include "tile_config.h"
// L2 eviction hints of the producers' 16-byte tile copies (0 none, 1 evict_last, 2 evict_first).  Measured at cfg4:
// D tiles evict_first (a D_pos tile is streamed once per sibling CTA and never again) +0.5 %; E tiles evict_last
// -0.4 %; both: no change; A tiles evict_first as well: -0.4 % (two more producer registers spill).
#ifndef SU2_HINT_E
#define SU2_HINT_E 0
#define SU2_HINT_D 2
#endif

namespace su2 {

namespace {

enum : int { PH_END = 1, PH_G2 = 2, PH_TRANS = 4 };

// One *phase* = a run of pipeline steps with regular addressing: the first product of one
// (task, position, T-chunk) -- nsteps stages of an A tile and an E tile, KS1 deep -- or its second
// product -- nsteps stages of a D tile.  Step s reads src + s * stride; both producers and consumers
// derive everything else (valid k extent, first/last flags) from s in registers.
struct PhaseDesc {
  const double* src0;   // first product: A tile origin of step 0;  second product: D tile origin
  const double* src1;   // first product: E tile origin of step 0
  double scale;         // coef * alpha_pos, applied when the first product parks T
  int stride0, stride1; // elements between consecutive steps
  int ld0, ld1;         // global leading dimensions
  int cval0;            // valid extent of tile 0 along c (rows of A / columns of F)
  int cval1;            // valid columns of the E tile (= width of the T chunk)
  int ktot;             // total k extent of the phase (k, or the chunk width)
  int nsteps;
  int flags;
  int pad;
};
constexpr int PHASE_RING = 16;  // producers run at most MAX_STAGE = 8 steps (hence phases) ahead of the consumers and write one more

struct GenState {       // iterator over the phases of one work item (shared memory; advanced by one thread)
  const double *A, *D, *E, *alpha;
  double coef, scale;
  int m, k, n, p, strideA, strideD, tflags;
  int u, u_end, pos, pos_end, chunk, nchunks, ncw_full, n0, ncw, phase, done;
  int row0, col0, rows_valid, cols_valid, nc_max;
};

__device__ __forceinline__ void gen_set_chunk(GenState& st) {
  st.n0 = st.chunk * st.ncw_full;
  st.ncw = min(st.ncw_full, st.n - st.n0);
  st.phase = 0;
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
  chunking(t.n, st.nc_max, st.nchunks, st.ncw_full);
  gen_set_pos(st);
}

// Emit the descriptor of the current phase and move to the next one.
__device__ __forceinline__ void gen_phase(GenState& st, PhaseDesc& d, const DevUnit* __restrict__ units,
                                          const DevTask* __restrict__ tasks, const double* __restrict__ psi) {
  if (st.done) {
    d.flags = PH_END;
    d.nsteps = 1;
    return;
  }
  if (st.phase == 0) {
    const bool tr = st.tflags & TASK_TRANS_A;
    d.src0 = st.A + (int64_t)st.pos * st.strideA + (tr ? (int64_t)st.row0 : (int64_t)st.row0 * st.k);
    d.stride0 = tr ? KS1 * st.m : KS1;
    d.ld0 = tr ? st.m : st.k;
    d.src1 = st.E + st.n0;
    d.stride1 = KS1 * st.n;
    d.ld1 = st.n;
    d.cval0 = st.rows_valid;
    d.cval1 = st.ncw;
    d.ktot = st.k;
    d.nsteps = (st.k + KS1 - 1) / KS1;
    d.scale = st.scale;
    d.flags = tr ? PH_TRANS : 0;
    st.phase = 1;
  } else {
    const bool tr = st.tflags & TASK_TRANS_D;
    d.src0 = st.D + (int64_t)st.pos * st.strideD +
             (tr ? (int64_t)st.n0 * st.p + st.col0 : (int64_t)st.col0 * st.n + st.n0);
    d.stride0 = tr ? KS2 * st.p : KS2;
    d.ld0 = tr ? st.p : st.n;
    d.cval0 = st.cols_valid;
    d.cval1 = 0;
    d.ktot = st.ncw;
    d.nsteps = (st.ncw + KS2 - 1) / KS2;
    d.flags = PH_G2 | (tr ? PH_TRANS : 0);
    if (++st.chunk < st.nchunks) gen_set_chunk(st);
    else if (++st.pos < st.pos_end) gen_set_pos(st);
    else if (++st.u < st.u_end) gen_load_unit(st, units, tasks, psi);
    else st.done = 1;
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

__device__ __forceinline__ void producer_bar() { asm volatile("bar.sync 2, 128;\n" ::: "memory"); }

// ---- staging: the four producer warps copy a quarter of every tile each ---------------------------
// Every tile lands in the same shared-memory layout, [j/4][j%4][c] with row stride CT+4 doubles
// (k-major k4 sub-tiles; CT+4 = 4 mod 8 makes the DMMA fragment loads conflict-free), so the math
// code does not depend on how the operator block is stored.  8-byte cp.async with zero fill: ragged
// block sizes and odd leading dimensions need no special cases.
// The copy loops are written with running addresses (one LDGSTS + two adds per element).
__device__ __forceinline__ void cp_async8_raw(unsigned dst, const void* src, int sz) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
// Source stored c-major, element (c, j) = src[c*ld + j]: 8 consecutive lanes read one 64-byte run, a warp
// instruction covers 4 rows; producer warp w takes the row groups  c/4 = w (mod 4).
constexpr int HINT_E = SU2_HINT_E, HINT_D = SU2_HINT_D;   // L2 eviction hints of the E / D tile copies
template <int CT, int KSX>
__device__ __forceinline__ void copy_cmajor(double* dst, const double* __restrict__ src, int ld, int cval, int jval,
                                            int w, int lane) {
  const int j = lane & 7, r = 4 * w + (lane >> 3);
  const int jpad = (jval + 3) & ~3;                  // the consumers read whole k4 sub-tiles
  const int cpad = (cval + 7) & ~7;
  unsigned d = smem_u32(dst + (j >> 2) * (4 * (CT + 4)) + (j & 3) * (CT + 4) + r);
  const char* s = reinterpret_cast<const char*>(src + (int64_t)r * ld + j);
  const int64_t sstep = (int64_t)ld * 128;           // sixteen rows further
#pragma unroll 1
  for (int c = r; c < cpad; c += 16) {               // rows beyond the block (fewer than 8) are zero-filled
    const bool rowok = c < cval;
#pragma unroll
    for (int g = 0; g < (KSX + 7) / 8; ++g)          // groups of 8 k columns = 2 sub-tiles = 8 (CT+4) doubles apart
      if (8 * g + j < jpad)
        cp_async8_raw(d + g * (8 * (CT + 4) * 8), rowok ? s + g * 64 : reinterpret_cast<const char*>(src),
                      (rowok && 8 * g + j < jval) ? 8 : 0);
    d += 128;
    s += sstep;
  }
}
// Source stored k-major, element (c, j) = src[j*ld + c]: runs along c are contiguous, so they move with
// 16-byte cp.async (half the LSU instructions of the 8-byte path: 19.7 vs 9.3 TB/s measured for this
// loop).  Rows are only 8-byte aligned (arbitrary block sizes), so a row whose first element sits at an
// odd double index is stored SHIFTED by one element in shared memory: element c lands at position
// c + parity, which makes every pair (c, c+1) with c = parity (mod 2) 16-byte aligned on both sides; the
// one element in front of the first pair is copied alone.  The consumers add the same parity to their
// fragment pointers (kmajor_shift).  A partial last pair uses src-size 8 (the rest is zero-filled), pairs
// beyond the block src-size 0.  Producer warp w takes the k rows j = w, w + 4, ...
__device__ __forceinline__ void cp_async16_raw(unsigned dst, const void* src, int sz) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ int addr_parity(const double* p) { return (int)((reinterpret_cast<uintptr_t>(p) >> 3) & 1u); }
// parity of row j = 4*sub + t (+ multiples of 4) of a k-major tile with origin `origin` and leading dimension ld
__device__ __forceinline__ int kmajor_shift(const double* origin, int ld, int t) {
  return (addr_parity(origin) ^ (t & ld)) & 1;
}
__device__ __forceinline__ void cp_async16_hint(unsigned dst, const void* src, int sz, uint64_t pol) {
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;\n" ::"r"(dst), "l"(src), "r"(sz), "l"(pol) : "memory");
}
// HINT: 0 = default L2 policy, 1 = evict_last (tile re-read by this and the sibling CTAs: E), 2 = evict_first
template <int CT, int HINT = 0>
__device__ __forceinline__ void copy_kmajor(double* dst, const double* __restrict__ src, int ld, int cval, int jval,
                                            int w, int lane) {
  uint64_t pol = 0;
  if (HINT == 1) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol));
  if (HINT == 2) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(pol));
  const int cpad = (cval + 7) & ~7;
  const int jpad = (jval + 3) & ~3;
  // The rows w, w+4, ... of this warp start at the same parity (4*ld is even) and their shared-memory rows
  // are one k4 sub-tile apart: everything but two running addresses is set up once per tile.
  const double* row = src + (int64_t)w * ld;
  const int pi = addr_parity(row);
  const int c0 = pi + 2 * lane;
  unsigned d0 = smem_u32(dst + w * (CT + 4)) + (unsigned)(c0 + pi) * 8u;      // this lane's first pair
  const char* s0 = reinterpret_cast<const char*>(row + c0);
  const int64_t rstep = (int64_t)ld * 32;                                      // four rows further (bytes)
#pragma unroll 1
  for (int j = w; j < jpad; j += 4) {
    const int lim = j < jval ? cval : 0;                       // rows beyond the k extent are zero
    if (pi && lane == 0) cp_async8_raw(d0 - 8, s0 - 8, lim > 0 ? 8 : 0);      // element 0 -> position 1
    unsigned d = d0;
    const char* s = s0;
#pragma unroll 2
    for (int c = c0; c < cpad; c += 64) {
      if (HINT) cp_async16_hint(d, s, min(16, max(0, (lim - c) * 8)), pol);
      else cp_async16_raw(d, s, min(16, max(0, (lim - c) * 8)));
      d += 512;
      s += 512;
    }
    d0 += 4 * (CT + 4) * 8;
    s0 += rstep;
  }
}

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}

// One pipeline stage (nsub <= NSUB k4 sub-steps) of a warp-level product: c[ii][j] += A_frag[ii] B_frag[j]
// for 4 m8-tiles (the first mt active) and NT n8-tiles.  a / b point at this lane's element of the
// first fragment; A_I / A_SUB / B_SUB are the compile-time strides between m8-tiles / k4 sub-steps
// (n8-tiles are 8 doubles apart).
template <int NSUB, int NT, int NACC, int A_I, int A_SUB, int B_SUB>
__device__ __forceinline__ void mma_stage(double (&c)[4][NACC][2], const double* __restrict__ a,
                                          const double* __restrict__ b, int nsub, int mt) {
  if (mt == 4 && nsub == NSUB) {
    // full stage: one straight-line block, so that the fragment loads of sub-step s+1 can be scheduled
    // under the DMMAs of sub-step s
#pragma unroll
    for (int sub = 0; sub < NSUB; ++sub) {
      double af[4], bf[NT];
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) af[ii] = a[sub * A_SUB + ii * A_I];
#pragma unroll
      for (int j = 0; j < NT; ++j) bf[j] = b[sub * B_SUB + j * 8];
#pragma unroll
      for (int j = 0; j < NT; ++j)
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) dmma(c[ii][j], af[ii], bf[j]);
    }
    return;
  }
#pragma unroll
  for (int sub = 0; sub < NSUB; ++sub) {
    if (sub < nsub) {
      double af[4], bf[NT];
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) af[ii] = a[sub * A_SUB + ii * A_I];
#pragma unroll
      for (int j = 0; j < NT; ++j) bf[j] = b[sub * B_SUB + j * 8];
#pragma unroll
      for (int j = 0; j < NT; ++j)
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
          if (ii < mt) dmma(c[ii][j], af[ii], bf[j]);
    }
  }
}


// ---- producer warps: all four walk every step and copy a quarter of its tiles -------------------------
// Warp 0 / lane 0 also runs the phase iterator, one phase ahead, into the descriptor ring.
template <int WR>
__device__ __forceinline__ void producer_item(const DevWork* __restrict__ wkp, const DevUnit* __restrict__ units,
                                              const DevTask* __restrict__ tasks, const double* __restrict__ psi,
                                              double* smem, GenState& st, PhaseDesc* pring, uint64_t* full,
                                              uint64_t* empty, int w, int lane) {
  using C = TileCfg<WR>;
  constexpr int NS = C::NSTAGE;
  double* stages = smem + C::TM * C::LDT;
  const bool gen = (w == 0 && lane == 0);
  if (gen) {
    const DevWork wk = *wkp;
    st.u = wk.unit0; st.u_end = wk.unit1; st.done = 0;
    st.row0 = wk.row0; st.col0 = wk.col0;
    st.rows_valid = min(C::TM, wk.m - wk.row0);
    st.cols_valid = min(C::TP, wk.p - wk.col0);
    st.nc_max = C::NC;
    if (st.u < st.u_end) gen_load_unit(st, units, tasks, psi);
    else st.done = 1;
    gen_phase(st, pring[0], units, tasks, psi);
  }
  unsigned pq = 0;
  int b = 0, par = 0;                                  // stage buffer and its fill parity
#pragma unroll 1
  for (;;) {
    producer_bar();                                     // descriptor pq is visible to the four producer warps
    // Phase constants are re-read from shared memory every step (volatile: LDS, ~30 cycles) instead of
    // being held in the 56 producer registers, where they would spill to local memory.
    const volatile PhaseDesc& d = pring[pq & (PHASE_RING - 1)];
    const int flags = d.flags, nsteps = d.nsteps;
#pragma unroll 1
    for (int s = 0; s < nsteps; ++s) {
      mbar_wait(&empty[b], par ^ 1);                    // consumers have released the previous fill
      if (!(flags & PH_END)) {
        double* stage = stages + b * C::STAGE;
        const double* src0 = d.src0 + (int64_t)s * d.stride0;
        if (!(flags & PH_G2)) {
          const int jval = min(KS1, d.ktot - s * KS1);
          if (flags & PH_TRANS) {
            copy_kmajor<C::TM>(stage, src0, d.ld0, d.cval0, jval, w, lane);
          } else {
            copy_cmajor<C::TM, KS1>(stage, src0, d.ld0, d.cval0, jval, w, lane);
          }
          copy_kmajor<C::NC, HINT_E>(stage + C::A_SZ, d.src1 + (int64_t)s * d.stride1, d.ld1, d.cval1, jval, w, lane);
        } else {
          const int jval = min(KS2, d.ktot - s * KS2);
          if (flags & PH_TRANS) copy_kmajor<C::TP, HINT_D>(stage, src0, d.ld0, d.cval0, jval, w, lane);
          else {
            copy_cmajor<C::TP, KS2>(stage, src0, d.ld0, d.cval0, jval, w, lane);
          }
        }
      }
      cp_async_mbar_arrive(&full[b]);          // 128 deferred arrivals: this lane's copies have landed
      if (w == 0) {
        __syncwarp();
        if (lane == 0) mbar_arrive(&full[b]);  // +1 (release): the phase descriptor is visible
      }
      if (++b == NS) { b = 0; par ^= 1; }
      if (s == 0 && gen && !(flags & PH_END))  // next phase's descriptor, while this step is in flight
        gen_phase(st, pring[(pq + 1) & (PHASE_RING - 1)], units, tasks, psi);
    }
    if (flags & PH_END) break;
    ++pq;
  }
}

// ---- consumer warps: LDS + DMMA only ------------------------------------------------------------------
// All steps of one phase for one warp: wait for the stage, multiply, release the stage.
// G2 = false: A fragments come from the stage (a_off inside it); G2 = true: from T (a_off + s*KS2).
template <int NS, int STAGE, bool G2, int NT, int NACC, int A_I, int A_SUB, int B_SUB>
__device__ __forceinline__ void run_phase(double (&c)[4][NACC][2], const double* stages, const double* Ts, int a_off,
                                          int b_off, int nsteps, int ktot, int mt, int& b, int& par, uint64_t* full,
                                          uint64_t* empty, int lane) {
  constexpr int KSX = G2 ? KS2 : KS1;
#pragma unroll 1
  for (int s = 0; s < nsteps; ++s) {
    if (s > 0) mbar_wait(&full[b], par);                        // step 0 was awaited by the caller
    if (NT > 0 && mt > 0) {
      const double* stage = stages + b * STAGE;
      const double* a = G2 ? Ts + a_off + s * KSX : stage + a_off;
      const int nsub = (min(KSX, ktot - s * KSX) + 3) >> 2;
      mma_stage<KSX / 4, (NT > 0 ? NT : 1), NACC, A_I, A_SUB, B_SUB>(c, a, stage + b_off, nsub, mt);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[b]);                      // stage released
    if (++b == NS) { b = 0; par ^= 1; }
  }
}

template <int WR>
__device__ __forceinline__ void consumer_item(const DevWork* __restrict__ wkp, double* __restrict__ out,
                                              double* __restrict__ partial, double* smem, const PhaseDesc* pring,
                                              uint64_t* full, uint64_t* empty, int cw, int lane) {
  using C = TileCfg<WR>;
  constexpr int WC = C::WC, TM = C::TM, TP = C::TP, NC = C::NC, LDT = C::LDT, LDE = NC + 4, NS = C::NSTAGE, ST = C::STAGE;
  const int g = lane >> 2, t = lane & 3;
  const int wr = cw / WC, wc = cw % WC;
  double* Ts = smem;
  const double* stages = smem + TM * LDT;

  const int rows_valid = min(TM, wkp->m - wkp->row0);
  const int cols_valid = min(TP, wkp->p - wkp->col0);
  const int mt = max(0, min(4, (rows_valid - wr * 32 + 7) >> 3));          // active m8-tiles of this warp
  const int ntiles2 = (cols_valid + 7) >> 3;
  const int ntw2 = (ntiles2 + WC - 1) / WC;
  const int ctile0 = wc * ntw2;
  const int nt2 = max(0, min(ntw2, ntiles2 - ctile0));                     // active n8-tiles (second product)
  const int a1_off = t * (TM + 4) + wr * 32 + g;                            // A fragment inside a stage
  const int t_off = (wr * 32 + g) * LDT + t;                                // A fragment of the second product inside T
  const int d_off = t * (TP + 4) + ctile0 * 8 + g;                          // D fragment inside a stage

  double acc[4][NT2][2];
  double tacc[4][NT1][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < NT2; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  unsigned cq = 0;
  int b = 0, par = 0;                                    // stage buffer and its fill parity
#pragma unroll 1
  for (;;) {
    mbar_wait(&full[b], par);                            // first step of the phase: its descriptor is visible too
    const PhaseDesc& d = pring[cq & (PHASE_RING - 1)];
    const int flags = d.flags, nsteps = d.nsteps, ktot = d.ktot;
    if (flags & PH_END) {
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[b]);
      break;
    }
    if (!(flags & PH_G2)) {
      // ---- first product: tacc (32 x 8 NT1 per warp) = A_pos[rows, :] E[:, chunk] ----------------
      const int ntiles1 = (d.cval1 + 7) >> 3;
      const int nt1w = (ntiles1 + WC - 1) / WC;
      const int tile0 = wc * nt1w;
      const int nt1 = max(0, min(nt1w, ntiles1 - tile0));
      const double sc = d.scale;
      const int e_off = C::A_SZ + t * LDE + tile0 * 8 + g + kmajor_shift(d.src1, d.ld1, t);
      const int a_off = a1_off + ((flags & PH_TRANS) ? kmajor_shift(d.src0, d.ld0, t) : 0);
#pragma unroll
      for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int j = 0; j < NT1; ++j) tacc[ii][j][0] = tacc[ii][j][1] = 0.0;
      switch (nt1) {
        case 1: run_phase<NS, ST, false, 1, NT1, 8, 4 * (TM + 4), 4 * LDE>(tacc, stages, Ts, a_off, e_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 2: run_phase<NS, ST, false, 2, NT1, 8, 4 * (TM + 4), 4 * LDE>(tacc, stages, Ts, a_off, e_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 3: run_phase<NS, ST, false, 3, NT1, 8, 4 * (TM + 4), 4 * LDE>(tacc, stages, Ts, a_off, e_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        default: run_phase<NS, ST, false, 0, NT1, 8, 4 * (TM + 4), 4 * LDE>(tacc, stages, Ts, a_off, e_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
      }
      consumer_bar();                              // every warp is done reading the previous T chunk
      double* trow = Ts + (wr * 32 + g) * LDT + tile0 * 8 + 2 * t;
#pragma unroll
      for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int j = 0; j < NT1; ++j)
          if (ii < mt && j < nt1)
            *reinterpret_cast<double2*>(trow + ii * 8 * LDT + j * 8) = make_double2(sc * tacc[ii][j][0], sc * tacc[ii][j][1]);
      consumer_bar();                              // the new T chunk is visible to every warp
    } else {
      // ---- second product: acc (32 x 8 NT2 per warp) += T_chunk D_pos[cols, chunk]^T --------------
      const int dd_off = d_off + ((flags & PH_TRANS) ? kmajor_shift(d.src0, d.ld0, t) : 0);
      switch (nt2) {
        case 1: run_phase<NS, ST, true, 1, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 2: run_phase<NS, ST, true, 2, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 3: run_phase<NS, ST, true, 3, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 4: run_phase<NS, ST, true, 4, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 5: run_phase<NS, ST, true, 5, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 6: run_phase<NS, ST, true, 6, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 7: run_phase<NS, ST, true, 7, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 8: run_phase<NS, ST, true, 8, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        case 9: run_phase<NS, ST, true, 9, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
        default: run_phase<NS, ST, true, 0, NT2, 8 * LDT, 4, 4 * (TP + 4)>(acc, stages, Ts, t_off, dd_off, nsteps, ktot, mt, b, par, full, empty, lane); break;
      }
    }
    ++cq;
  }

  // ---- epilogue: the tile leaves the registers once per work item -----------------------------
  const DevWork wk = *wkp;            // re-read here: nothing of it stays live across the item
  double* dst = ((wk.to_partial & 1) ? partial : out) + wk.dst_off;
  const bool accumulate = wk.to_partial & 2;
#pragma unroll
  for (int ii = 0; ii < 4; ++ii)
#pragma unroll
    for (int j = 0; j < NT2; ++j)
      if (ii < mt && j < nt2) {
        const int r = wk.row0 + wr * 32 + ii * 8 + g;
        const int q = wk.col0 + (ctile0 + j) * 8 + 2 * t;
        if (r < wk.m) {
          double* o = dst + (int64_t)r * wk.p + q;
          if (q < wk.p) o[0] = accumulate ? o[0] + acc[ii][j][0] : acc[ii][j][0];
          if (q + 1 < wk.p) o[1] = accumulate ? o[1] + acc[ii][j][1] : acc[ii][j][1];
        }
      }
}

__global__ void __launch_bounds__(NTHREADS, 1)
heff_dmma_kernel(const DevWork* __restrict__ work, int nwork, const DevUnit* __restrict__ units,
                 const DevTask* __restrict__ tasks, const double* __restrict__ psi, double* __restrict__ out,
                 double* __restrict__ partial, int* __restrict__ counter) {
  extern __shared__ __align__(16) double smem[];
  __shared__ GenState gs;
  __shared__ PhaseDesc pring[PHASE_RING];
  __shared__ __align__(8) uint64_t full[MAX_STAGE];
  __shared__ __align__(8) uint64_t empty[MAX_STAGE];
  __shared__ int s_w;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (warp < NPRODUCERS) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;\n");
#pragma unroll 1
    for (;;) {
      cta_bar();                         // previous item retired: pipeline drained, barriers idle
      if (tid == 0) {
        s_w = atomicAdd(counter, 1);
        for (int i = 0; i < MAX_STAGE; ++i) {
          mbar_init(&full[i], NPRODUCERS * 32 + 1);   // deferred cp.async arrivals of every producer lane + the descriptor writer
          mbar_init(&empty[i], NWARPS);               // one arrival per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
      }
      cta_bar();
      const int w = s_w;
      if (w >= nwork) break;
      const int wr = work[w].wr;
      if (wr == 1) producer_item<1>(work + w, units, tasks, psi, smem, gs, pring, full, empty, warp, lane);
      else if (wr == 2) producer_item<2>(work + w, units, tasks, psi, smem, gs, pring, full, empty, warp, lane);
      else producer_item<4>(work + w, units, tasks, psi, smem, gs, pring, full, empty, warp, lane);
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 224;\n");
    const int cw = warp - NPRODUCERS;
#pragma unroll 1
    for (;;) {
      cta_bar();
      cta_bar();
      const int w = s_w;
      if (w >= nwork) break;
      const int wr = work[w].wr;
      if (wr == 1) consumer_item<1>(work + w, out, partial, smem, pring, full, empty, cw, lane);
      else if (wr == 2) consumer_item<2>(work + w, out, partial, smem, pring, full, empty, cw, lane);
      else consumer_item<4>(work + w, out, partial, smem, pring, full, empty, cw, lane);
    }
  }
}

}  // namespace

su2_status launch_heff_dmma_tables(const DevWork* work, int nwork, const DevUnit* units, const DevTask* tasks, const double* psi,
                                   double* out, double* partial, int* counter, int num_sms, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  if (nwork == 0) return SU2_OK;
  static bool attr_set = false;
  const size_t smem_bytes = (size_t)SMEM_DOUBLES_MAX * sizeof(double);
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(heff_dmma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) { set_cuda_error("cudaFuncSetAttribute(heff_dmma_kernel)", (int)e); return SU2_ERR_CUDA; }
    attr_set = true;
  }
  const int grid = std::min(nwork, num_sms);
  heff_dmma_kernel<<<grid, NTHREADS, smem_bytes, stream>>>(work, nwork, units, tasks, psi, out, partial, counter);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_cuda_error("heff_dmma_kernel launch", (int)e); return SU2_ERR_CUDA; }
  count_launch();
  return SU2_OK;
}

su2_status launch_heff_dmma(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream_v) {
  return launch_heff_dmma_tables(plan->d_work, (int)plan->h_work.size(), plan->d_units, plan->d_tasks, psi, out, partial,
                                 plan->d_counter, plan->num_sms, stream_v);
}

}  // namespace su2
