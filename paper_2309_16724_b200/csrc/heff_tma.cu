// sm_100a fused GEMM-pair kernel of the hot path:
//
//   F_tile (TM x TP, registers) += sum_{task, pos} (coef alpha_pos) * (A_pos[rows,:] E) D_pos[cols,:]^T
//
// the paper's two SBGEMM steps fused per task: the intermediate T = A_pos E never leaves the SM
// (accumulated in registers, parked in shared memory as the A operand of the second product), and the sum over
// positions is the K loop of the second product (the paper's stripe trick).
//
// Arithmetic: FP64 tensor instructions mma.sync.aligned.m8n8k4.f64 (SASS DMMA.8x8x4) -- the only FP64 matrix
// instruction sm_100a exposes (tcgen05 has no f64 kind); measured at 37.1 TFLOP/s = 99.8 % of
// 148 SM x 64 FMA/clk x 1.965 GHz, against 33.8 TFLOP/s for a DFMA loop (profiles/r01_fp64_peak_probe.txt).
//
// Structure.  Persistent CTAs (one per SM) pull work items (segment x output tile) from an atomic queue in the
// plan's longest-first order.  Every (task, position, T-chunk) of an item is a pair of *phases*: the first product
// (stages of an A box + E boxes, KS1 deep) and the second product (stages of D boxes, KS2 deep).
//   * ONE elected thread of the producer warpgroup (40 registers after setmaxnreg.dec) walks the phases: it waits
//     for a stage's "empty" mbarrier, posts the stage's byte count on its "full" mbarrier (arrive.expect_tx) and
//     issues the stage's bulk-tensor copies (cp.async.bulk.tensor.3d, SASS UTMALDG).  Ragged block edges, odd
//     extents and the k tails are the TMA unit's out-of-bounds zero fill: there is not one predicate on the load
//     side.  All boxes land with a row pitch of 4 (mod 8) doubles (tile_config.h), so the m8n8k4 fragment loads are
//     conflict-free without swizzling, for blocks used as stored and for blocks read transposed alike.
//   * warps 4-15 (three warpgroups, 152 registers after setmaxnreg.inc; three warps per SM sub-partition, which is
//     what hides the fixed issue cadence of DMMA.8x8x4) are CONSUMERS: wait on the stage's "full" mbarrier, LDS +
//     DMMA with register-double-buffered fragments, release the stage on its "empty" mbarrier.  The T hand-over
//     between the two products uses a named barrier of the 384 consumer threads.
// The phase stream is continuous across work items of one tile class: the producer fetches the next item while the
// consumers still work on the current one, so the pipeline does not drain at item boundaries (it does when the
// tile class changes, because the stage geometry changes).
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>

#include "su2_internal.h"
#include "tile_config.h"

namespace su2 {

namespace {

enum : int { PH_END = 1, PH_G2 = 2, PH_TRANS = 4, PH_FIRST = 8, PH_LAST = 16, PH_RESET = 32, PH_NOBAR = 64 };

// Consumer-visible part of one phase (ring in shared memory, written by the producer thread one or more phases
// ahead; made visible by the release/acquire pair on the "full" mbarrier of the phase's first stage).
struct PhaseInfo {
  double scale;     // coef * alpha_pos, applied when the first product parks T
  int flags;
  int nsteps;       // pipeline stages of this phase
  int ktot;         // k extent of the phase (k of the task, or the width of the T chunk)
  int ncw;          // first product: columns of the T chunk
  int work;         // PH_FIRST: index of the work item that starts here
  int pad;
};
constexpr int PHASE_RING = 16;     // the producer runs at most MAX_STAGE stages (hence phases) ahead, and writes one more
#ifndef SU2_PRODUCER_REGS
#define SU2_PRODUCER_REGS 40
#define SU2_CONSUMER_REGS 152
#endif
constexpr int PRODUCER_REGS = SU2_PRODUCER_REGS, CONSUMER_REGS = SU2_CONSUMER_REGS;
static_assert(NPRODUCERS * 32 * PRODUCER_REGS + NWARPS * 32 * CONSUMER_REGS <= 65536, "register file");

// ---- PTX helpers -------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
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
__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;\n" ::"n"(NWARPS * 32) : "memory"); }

// One box of a rank-3 tensor map {columns, rows, items} -> shared memory; completion is counted in bytes on `bar`.
__device__ __forceinline__ void tma_box(unsigned dst, const void* map, int c0, int c1, int c2, uint64_t* bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;\n"
      ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

// L2 eviction priority of the A / D / E boxes (0 evict_normal, 1 evict_last, 2 evict_first).  Measured at cfg4's block sizes
// (DESIGN.md section 7): the apply time is the same for every combination (the kernel is not bound by its loads); DRAM
// reads are lowest with E evict_last (every sibling CTA and every position re-reads it) and A, D left alone --
// evict_first on the D boxes, round 1's choice, costs 20 % more DRAM traffic here because sibling row-tile CTAs arrive late.
#ifndef SU2_GANG_AHEAD
#define SU2_GANG_AHEAD 2      // positions a gang member may run in front of a running member behind it (< 0: no pacing)
#define SU2_GANG_NEAR 48      // members further behind than this are another wave of the queue: ignored
#endif
#ifndef SU2_POL_A
#define SU2_POL_A 0
#define SU2_POL_D 0
#define SU2_POL_E 1
#endif
template <int KIND>
__device__ __forceinline__ uint64_t l2_policy() {
  uint64_t pol;
  if (KIND == 1) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol));
  else if (KIND == 2) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(pol));
  else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;\n" : "=l"(pol));
  return pol;
}

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}

// ---- the producer thread --------------------------------------------------------------------------------------
struct Pipe {          // position in the stage ring; one parity bit per barrier (the ring length depends on the class)
  int b;
  unsigned par;
  unsigned pq;         // phases emitted / consumed
};

template <int WR>
__device__ __forceinline__ void produce_item(const DevWork& wk, int w, bool reset, const DevUnit* __restrict__ units,
                                             const DevTask* __restrict__ tasks, const CUtensorMap* __restrict__ maps,
                                             unsigned stage0, PhaseInfo* ring, uint64_t* full, uint64_t* empty, Pipe& pp,
                                             uint64_t pol_a, uint64_t pol_d, uint64_t pol_e, int* __restrict__ gangs) {
  using C = TileCfg<WR>;
  constexpr int NS = C::NSTAGE;
  constexpr int NEB = C::NEBOX, NDB = C::NDBOX;
  constexpr unsigned E_BYTES = NEB * EBOX_SZ * 8u;
  bool first = true;
  // Pacing of a gang: the row tiles of one (sector, segment, column tile) walk through the same tasks and positions and read
  // the same D_pos and E boxes.  Left alone they drift apart by more positions than their share of L2 holds and every one of
  // them streams D from DRAM again (68 % of the DRAM reads, profiles/r02_traffic_cfg4.md).  Each member publishes the number
  // of positions it has issued; a member more than GANG_AHEAD positions in front of another RUNNING member that is less than
  // GANG_NEAR behind holds its loads until that one has caught up.  Members that started much later (another wave of the
  // queue) are out of reach of L2 anyway and are ignored; finished members publish INT_MAX.  Nobody waits for a member that
  // has not started, and the hindmost running member never waits: no deadlock.  Only this thread (the producer) polls.
  constexpr int GANG_AHEAD = SU2_GANG_AHEAD, GANG_NEAR = SU2_GANG_NEAR;
  volatile int* gang = (GANG_AHEAD >= 0 && gangs != nullptr && wk.gang >= 0) ? gangs + wk.gang : nullptr;
  const int gang_n = wk.m / C::TM, gang_me = wk.row0 / C::TM;      // full row tiles only (plan.cpp)
  int gang_step = 0;
#pragma unroll 1
  for (int u = wk.unit0; u < wk.unit1; ++u) {
    const DevUnit un = units[u];
    const DevTask* __restrict__ t = tasks + un.task;
    const int k = t->k, n = t->n;
    const unsigned tflags = t->flags;
    const double coef = t->coef;
    const double* __restrict__ alpha = t->alpha;
    const CUtensorMap* mA = maps + t->mapA;
    const CUtensorMap* mD = maps + t->mapD;
    const CUtensorMap* mE = maps + t->mapE;
    const int e_item = t->e_item;
    const int posA = t->strideA ? 1 : 0, posD = t->strideD ? 1 : 0;   // a block shared by all positions has one item
    int nchunks, ncw_full;
    chunking(n, C::NC, nchunks, ncw_full);
    const int nsteps1 = (k + KS1 - 1) / KS1;
    const unsigned a_bytes = (tflags & TASK_TRANS_A) ? (unsigned)(KS1 * (C::TM + 4) * 8) : (unsigned)(C::TM * KS1 * 8);
    const unsigned d_bytes = NDB * ((tflags & TASK_TRANS_D) ? (unsigned)(KS2 * DBOX_LD * 8) : (unsigned)(DBOX_C * KS2 * 8));
#pragma unroll 1
    for (int pos = un.pos0; pos < un.pos1; ++pos) {
      const double scale = coef * (alpha ? alpha[pos] : 1.0);
      if (gang) {
        gang[gang_me] = gang_step;
        for (;;) {
          bool hold = false;
          for (int j = 0; j < gang_n; ++j) {
            const int pj = gang[j];
            if (pj >= 0 && pj < gang_step - GANG_AHEAD && pj > gang_step - GANG_NEAR) { hold = true; break; }
          }
          if (!hold) break;
          __nanosleep(500);
        }
        ++gang_step;
      }
#pragma unroll 1
      for (int chunk = 0; chunk < nchunks; ++chunk) {
        const int n0 = chunk * ncw_full;
        const int ncw = min(ncw_full, n - n0);
        // ---- first product: T chunk = A_pos[rows, :] E[:, n0 .. n0 + ncw)
        {
          PhaseInfo& pi = ring[pp.pq & (PHASE_RING - 1)];
          pi.scale = scale;
          // No barrier is needed in front of the T store when the first product has at least NS stages: its stage NS-1
          // refills the ring slot of the LAST stage of the previous second product, and a slot is refilled only after all
          // twelve warps have released it -- so a warp that has consumed the whole first product knows that every warp has
          // left the previous second product (has stopped reading T)
          pi.flags = ((tflags & TASK_TRANS_A) ? PH_TRANS : 0) | (first ? PH_FIRST : 0) | ((nsteps1 >= NS && !first) ? PH_NOBAR : 0);
          pi.nsteps = nsteps1;
          pi.ktot = k;
          pi.ncw = ncw;
          pi.work = w;
          first = false;
#pragma unroll 1
          for (int s = 0; s < nsteps1; ++s) {
            const int b = pp.b;
            mbar_wait(&empty[b], ((pp.par >> b) & 1) ^ 1);          // consumers have released the previous fill
            mbar_arrive_expect_tx(&full[b], a_bytes + E_BYTES);     // (release: the phase record is visible)
            const unsigned st = stage0 + (unsigned)b * (C::STAGE * 8u);
            const int k0 = s * KS1;
            if (tflags & TASK_TRANS_A) tma_box(st, mA, wk.row0, k0, pos * posA, &full[b], pol_a);
            else tma_box(st, mA, k0, wk.row0, pos * posA, &full[b], pol_a);
#pragma unroll
            for (int e = 0; e < NEB; ++e)
              tma_box(st + (unsigned)(C::A_SZ + e * EBOX_SZ) * 8u, mE, n0 + e * EBOX_C, k0, e_item, &full[b], pol_e);
            pp.par ^= 1u << b;
            pp.b = (b + 1 == NS) ? 0 : b + 1;
          }
          ++pp.pq;
        }
        // ---- second product: F_tile += T chunk D_pos[cols, n0 .. n0 + ncw)^T
        {
          const bool last = (chunk + 1 == nchunks) && (pos + 1 == un.pos1) && (u + 1 == wk.unit1);
          const int nsteps2 = (ncw + KS2 - 1) / KS2;
          PhaseInfo& pi = ring[pp.pq & (PHASE_RING - 1)];
          pi.scale = 0.0;
          pi.flags = PH_G2 | ((tflags & TASK_TRANS_D) ? PH_TRANS : 0) | (last ? PH_LAST : 0) | ((last && reset) ? PH_RESET : 0);
          pi.nsteps = nsteps2;
          pi.ktot = ncw;
          pi.ncw = 0;
          pi.work = w;
#pragma unroll 1
          for (int s = 0; s < nsteps2; ++s) {
            const int b = pp.b;
            mbar_wait(&empty[b], ((pp.par >> b) & 1) ^ 1);
            mbar_arrive_expect_tx(&full[b], d_bytes);
            const unsigned st = stage0 + (unsigned)b * (C::STAGE * 8u);
            const int kk = n0 + s * KS2;
#pragma unroll
            for (int d = 0; d < NDB; ++d) {
              if (tflags & TASK_TRANS_D) tma_box(st + (unsigned)(d * DBOX_SZ) * 8u, mD, wk.col0 + d * DBOX_C, kk, pos * posD, &full[b], pol_d);
              else tma_box(st + (unsigned)(d * DBOX_SZ) * 8u, mD, kk, wk.col0 + d * DBOX_C, pos * posD, &full[b], pol_d);
            }
            pp.par ^= 1u << b;
            pp.b = (b + 1 == NS) ? 0 : b + 1;
          }
          ++pp.pq;
        }
      }
    }
  }
  if (gang) gang[gang_me] = 0x7fffffff;          // finished: out of every member's window
}

template <int MT, int NT, int NACC, int A_I, int A_SUB, int B_J, int B_SUB>
__device__ __forceinline__ void mma_ragged(double (&c)[4][NACC][2], const double* __restrict__ a,
                                           const double* __restrict__ b, int nsub) {
#pragma unroll 1
  for (int sub = 0; sub < nsub; ++sub) {
    double af[MT], bf[NT];
#pragma unroll
    for (int ii = 0; ii < MT; ++ii) af[ii] = a[sub * A_SUB + ii * A_I];
#pragma unroll
    for (int j = 0; j < NT; ++j) bf[j] = b[sub * B_SUB + j * B_J];
#pragma unroll
    for (int j = 0; j < NT; ++j)
#pragma unroll
      for (int ii = 0; ii < MT; ++ii) dmma(c[ii][j], af[ii], bf[j]);
  }
}

// One pipeline stage (nsub <= NSUB k4 sub-steps) of a warp-level product: c[ii][j] += A_frag[ii] B_frag[j] for
// 4 m8-tiles (the first mt active) and NT n8-tiles.  a / b point at this lane's element of the first fragment;
// A_I / B_J are the strides between m8-tiles / n8-tiles, A_SUB / B_SUB between k4 sub-steps.
template <int NSUB, int NT, int NACC, int A_I, int A_SUB, int B_J, int B_SUB>
__device__ __forceinline__ void mma_stage(double (&c)[4][NACC][2], const double* __restrict__ a,
                                          const double* __restrict__ b, int nsub, int mt) {
  if (mt == 4 && nsub == NSUB) {
    // full stage: straight-line, fragments of sub-step s+1 are loaded into a second register set under the DMMAs
    // of sub-step s (ptxas keeps only part of that distance; with three warps per sub-partition the rest is covered)
    double af[2][4], bf[2][NT];
#pragma unroll
    for (int ii = 0; ii < 4; ++ii) af[0][ii] = a[ii * A_I];
#pragma unroll
    for (int j = 0; j < NT; ++j) bf[0][j] = b[j * B_J];
#pragma unroll
    for (int sub = 0; sub < NSUB; ++sub) {
      const int cur = sub & 1, nxt = cur ^ 1;
      if (sub + 1 < NSUB) {
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) af[nxt][ii] = a[(sub + 1) * A_SUB + ii * A_I];
#pragma unroll
        for (int j = 0; j < NT; ++j) bf[nxt][j] = b[(sub + 1) * B_SUB + j * B_J];
      }
#pragma unroll
      for (int j = 0; j < NT; ++j)
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) dmma(c[ii][j], af[cur][ii], bf[cur][j]);
    }
    return;
  }
  // ragged stage (k tail of a phase, or a row tile with fewer than 32 valid rows): rolled loop over the sub-steps,
  // instantiated per number of active m8-tiles -- a predicated-off DMMA still occupies its slot in the FP64 tensor pipe
  // (sm__ops_path_tensor_src_fp64 counts it), so `if (ii < mt) dmma(...)` made the last row tile of every sector pay
  // for four m8-tiles whatever it held
  switch (mt) {
    case 1: mma_ragged<1, NT, NACC, A_I, A_SUB, B_J, B_SUB>(c, a, b, nsub); break;
    case 2: mma_ragged<2, NT, NACC, A_I, A_SUB, B_J, B_SUB>(c, a, b, nsub); break;
    case 3: mma_ragged<3, NT, NACC, A_I, A_SUB, B_J, B_SUB>(c, a, b, nsub); break;
    default: mma_ragged<4, NT, NACC, A_I, A_SUB, B_J, B_SUB>(c, a, b, nsub); break;
  }
}

// ---- consumer warps: LDS + DMMA only ------------------------------------------------------------------
// All steps of one phase for one warp: wait for the stage, multiply, release the stage.
// G2 = false: A fragments come from the stage (a_off inside it); G2 = true: from T (a_off + s*KS2).
template <int NS, int STAGE, bool G2, int NT, int NACC, int A_I, int A_SUB, int B_J, int B_SUB>
__device__ __forceinline__ void run_phase(double (&c)[4][NACC][2], const double* stages, const double* Ts, int a_off,
                                          int b_off, int nsteps, int ktot, int mt, Pipe& cp, uint64_t* full,
                                          uint64_t* empty, int lane) {
  constexpr int KSX = G2 ? KS2 : KS1;
#pragma unroll 1
  for (int s = 0; s < nsteps; ++s) {
    const int b = cp.b;
    if (s > 0) mbar_wait(&full[b], (cp.par >> b) & 1);            // step 0 was awaited by the caller
    if (NT > 0 && mt > 0) {
      const double* stage = stages + b * STAGE;
      const double* a = G2 ? Ts + a_off + s * KSX : stage + a_off;
      const int nsub = (min(KSX, ktot - s * KSX) + 3) >> 2;
      mma_stage<KSX / 4, (NT > 0 ? NT : 1), NACC, A_I, A_SUB, B_J, B_SUB>(c, a, stage + b_off, nsub, mt);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[b]);                        // stage released
    cp.par ^= 1u << b;
    cp.b = (b + 1 == NS) ? 0 : b + 1;
  }
}

// One work item: phases from the PH_FIRST record `info` (whose first stage the caller has awaited) to the record
// flagged PH_LAST, then the epilogue.
template <int WR>
__device__ __forceinline__ void consume_item(PhaseInfo info, const DevWork* __restrict__ work, double* __restrict__ out,
                                             double* __restrict__ partial, double* smem, const PhaseInfo* ring,
                                             uint64_t* full, uint64_t* empty, Pipe& cp, int cw, int lane) {
  using C = TileCfg<WR>;
  constexpr int WC = C::WC, TM = C::TM, LDT = C::LDT, NS = C::NSTAGE, ST = C::STAGE;
  const int g = lane >> 2, t = lane & 3;
  const int wr = cw / WC, wc = cw % WC;
  double* Ts = smem;
  const double* stages = smem + C::T_SZ;

  const DevWork wk = work[info.work];
  const int rows_valid = min(TM, wk.m - wk.row0);
  const int cols_valid = min(C::TP, wk.p - wk.col0);
  const int mt = max(0, min(4, (rows_valid - wr * 32 + 7) >> 3));          // active m8-tiles of this warp
  const int nt2 = max(0, min(NT2, ((cols_valid + 7) >> 3) - wc * NT2));    // active n8-tiles (second product)
  const int a_c_off = (wr * 32 + g) * KS1 + t;                              // A fragment, block as stored (c-major box)
  const int a_k_off = t * (TM + 4) + wr * 32 + g;                           // A fragment, block read transposed
  const int e_off = C::A_SZ + (wc / WPB) * EBOX_SZ + t * EBOX_LD + (wc % WPB) * (8 * NT1) + g;
  const int t_off = (wr * 32 + g) * LDT + t;                                // A fragment of the second product inside T
  const int d_k_off = (wc / WPB) * DBOX_SZ + t * DBOX_LD + (wc % WPB) * (8 * NT2) + g;
  const int d_c_off = (wc / WPB) * DBOX_SZ + ((wc % WPB) * (8 * NT2) + g) * KS2 + t;

  double acc[4][NT2][2];
  double tacc[4][NT1][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < NT2; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll 1
  for (;;) {
    const int flags = info.flags, nsteps = info.nsteps, ktot = info.ktot;
    if (!(flags & PH_G2)) {
      // ---- first product: tacc (32 x 16 per warp) = A_pos[rows, :] E[:, chunk] ----------------
      const int nt1 = max(0, min(NT1, ((info.ncw + 7) >> 3) - wc * NT1));
      const double sc = info.scale;
#pragma unroll
      for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int j = 0; j < NT1; ++j) tacc[ii][j][0] = tacc[ii][j][1] = 0.0;
      if (flags & PH_TRANS) {
        switch (nt1) {
          case 1: run_phase<NS, ST, false, 1, NT1, 8, 4 * (TM + 4), 8, 4 * EBOX_LD>(tacc, stages, Ts, a_k_off, e_off, nsteps, ktot, mt, cp, full, empty, lane); break;
          case 2: run_phase<NS, ST, false, (2 <= NT1 ? 2 : 0), NT1, 8, 4 * (TM + 4), 8, 4 * EBOX_LD>(tacc, stages, Ts, a_k_off, e_off, nsteps, ktot, mt, cp, full, empty, lane); break;
          case 3: run_phase<NS, ST, false, (3 <= NT1 ? 3 : 0), NT1, 8, 4 * (TM + 4), 8, 4 * EBOX_LD>(tacc, stages, Ts, a_k_off, e_off, nsteps, ktot, mt, cp, full, empty, lane); break;
          default: run_phase<NS, ST, false, 0, NT1, 8, 4 * (TM + 4), 8, 4 * EBOX_LD>(tacc, stages, Ts, a_k_off, e_off, nsteps, ktot, mt, cp, full, empty, lane); break;
        }
      } else {
        switch (nt1) {
          case 1: run_phase<NS, ST, false, 1, NT1, 8 * KS1, 4, 8, 4 * EBOX_LD>(tacc, stages, Ts, a_c_off, e_off, nsteps, ktot, mt, cp, full, empty, lane); break;
          case 2: run_phase<NS, ST, false, (2 <= NT1 ? 2 : 0), NT1, 8 * KS1, 4, 8, 4 * EBOX_LD>(tacc, stages, Ts, a_c_off, e_off, nsteps, ktot, mt, cp, full, empty, lane); break;
          case 3: run_phase<NS, ST, false, (3 <= NT1 ? 3 : 0), NT1, 8 * KS1, 4, 8, 4 * EBOX_LD>(tacc, stages, Ts, a_c_off, e_off, nsteps, ktot, mt, cp, full, empty, lane); break;
          default: run_phase<NS, ST, false, 0, NT1, 8 * KS1, 4, 8, 4 * EBOX_LD>(tacc, stages, Ts, a_c_off, e_off, nsteps, ktot, mt, cp, full, empty, lane); break;
        }
      }
      if (!(flags & PH_NOBAR)) consumer_bar();     // every warp is done reading the previous T chunk
      double* trow = Ts + (wr * 32 + g) * LDT + wc * (8 * NT1) + 2 * t;
#pragma unroll
      for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int j = 0; j < NT1; ++j)
          if (ii < mt && j < nt1)
            *reinterpret_cast<double2*>(trow + ii * 8 * LDT + j * 8) = make_double2(sc * tacc[ii][j][0], sc * tacc[ii][j][1]);
      consumer_bar();                              // the new T chunk is visible to every warp
    } else {
      // ---- second product: acc (32 x 48 per warp) += T_chunk D_pos[cols, chunk]^T --------------
#define SU2_G2_CASES(AOFF, BJ, BSUB) \
      switch (nt2) { \
        case 1: run_phase<NS, ST, true, (1 <= NT2 ? 1 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        case 2: run_phase<NS, ST, true, (2 <= NT2 ? 2 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        case 3: run_phase<NS, ST, true, (3 <= NT2 ? 3 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        case 4: run_phase<NS, ST, true, (4 <= NT2 ? 4 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        case 5: run_phase<NS, ST, true, (5 <= NT2 ? 5 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        case 6: run_phase<NS, ST, true, (6 <= NT2 ? 6 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        case 7: run_phase<NS, ST, true, (7 <= NT2 ? 7 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        case 8: run_phase<NS, ST, true, (8 <= NT2 ? 8 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        case 9: run_phase<NS, ST, true, (9 <= NT2 ? 9 : 0), NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
        default: run_phase<NS, ST, true, 0, NT2, 8 * LDT, 4, BJ, BSUB>(acc, stages, Ts, t_off, AOFF, nsteps, ktot, mt, cp, full, empty, lane); break; \
      }
      if (flags & PH_TRANS) { SU2_G2_CASES(d_k_off, 8, 4 * DBOX_LD) }
      else { SU2_G2_CASES(d_c_off, 8 * KS2, 4) }
#undef SU2_G2_CASES
    }
    ++cp.pq;
    if (flags & PH_LAST) {
      if (flags & PH_RESET) cp.b = 0;              // the stream restarts at stage 0 (class change or end)
      break;
    }
    mbar_wait(&full[cp.b], (cp.par >> cp.b) & 1);  // first step of the next phase: its record is visible too
    info = ring[cp.pq & (PHASE_RING - 1)];
  }

  // ---- epilogue: the tile leaves the registers once per work item -----------------------------
  double* dst = ((wk.to_partial & 1) ? partial : out) + wk.dst_off;
  const bool accumulate = wk.to_partial & 2;
#pragma unroll
  for (int ii = 0; ii < 4; ++ii)
#pragma unroll
    for (int j = 0; j < NT2; ++j)
      if (ii < mt && j < nt2) {
        const int r = wk.row0 + wr * 32 + ii * 8 + g;
        const int q = wk.col0 + (wc * NT2 + j) * 8 + 2 * t;
        if (r < wk.m) {
          double* o = dst + (int64_t)r * wk.ldo + q;
          if (q < wk.p) o[0] = accumulate ? o[0] + acc[ii][j][0] : acc[ii][j][0];
          if (q + 1 < wk.p) o[1] = accumulate ? o[1] + acc[ii][j][1] : acc[ii][j][1];
        }
      }
}

__global__ void __launch_bounds__(NTHREADS, 1)
heff_tma_kernel(const DevWork* __restrict__ work, int nwork, const DevUnit* __restrict__ units,
                const DevTask* __restrict__ tasks, const CUtensorMap* __restrict__ maps, double* __restrict__ out,
                double* __restrict__ partial, int* __restrict__ counter, int* __restrict__ gangs) {
  extern __shared__ __align__(1024) double smem[];
  __shared__ PhaseInfo ring[PHASE_RING];
  __shared__ __align__(8) uint64_t full[MAX_STAGE];
  __shared__ __align__(8) uint64_t empty[MAX_STAGE];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    for (int i = 0; i < MAX_STAGE; ++i) {
      mbar_init(&full[i], 1);            // the producer's arrive.expect_tx; the bytes of the boxes complete the phase
      mbar_init(&empty[i], NWARPS);      // one arrival per consumer warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  if (warp < NPRODUCERS) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(PRODUCER_REGS));
    if (tid != 0) return;
    const uint64_t pol_a = l2_policy<SU2_POL_A>(), pol_d = l2_policy<SU2_POL_D>(), pol_e = l2_policy<SU2_POL_E>();
    Pipe pp{0, 0u, 0u};
    int w = atomicAdd(counter, 1);
#pragma unroll 1
    for (;;) {
      if (w >= nwork) {                  // end of the stream; the ring position is 0 here (start, or after a reset)
        ring[pp.pq & (PHASE_RING - 1)].flags = PH_END;
        mbar_arrive(&full[0]);
        break;
      }
      const DevWork wk = work[w];
      // the next item is claimed one item ahead: the last phase of this item tells the consumers whether the
      // stream continues on the running stage (same tile class) or restarts at stage 0 (class change, end)
      const int wn = atomicAdd(counter, 1);
      const bool reset = wn >= nwork || work[wn].wr != wk.wr;
      const unsigned stage0 = smem_u32(smem + (wk.wr == 1 ? TileCfg<1>::T_SZ : wk.wr == 2 ? TileCfg<2>::T_SZ : TileCfg<4>::T_SZ));
      if (wk.wr == 1) produce_item<1>(wk, w, reset, units, tasks, maps, stage0, ring, full, empty, pp, pol_a, pol_d, pol_e, gangs);
      else if (wk.wr == 2) produce_item<2>(wk, w, reset, units, tasks, maps, stage0, ring, full, empty, pp, pol_a, pol_d, pol_e, gangs);
      else produce_item<4>(wk, w, reset, units, tasks, maps, stage0, ring, full, empty, pp, pol_a, pol_d, pol_e, gangs);
      if (reset) {
        // the stage geometry changes (or the stream ends): wait until every stage in flight has been released
        for (int i = 0; i < MAX_STAGE; ++i) mbar_wait(&empty[i], ((pp.par >> i) & 1) ^ 1);
        pp.b = 0;
      }
      w = wn;
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(CONSUMER_REGS));
    const int cw = warp - NPRODUCERS;
    Pipe cp{0, 0u, 0u};
#pragma unroll 1
    for (;;) {
      mbar_wait(&full[cp.b], (cp.par >> cp.b) & 1);      // first stage of the next item (or the end record)
      const PhaseInfo info = ring[cp.pq & (PHASE_RING - 1)];
      if (info.flags & PH_END) break;
      const int wr = work[info.work].wr;
      if (wr == 1) consume_item<1>(info, work, out, partial, smem, ring, full, empty, cp, cw, lane);
      else if (wr == 2) consume_item<2>(info, work, out, partial, smem, ring, full, empty, cp, cw, lane);
      else consume_item<4>(info, work, out, partial, smem, ring, full, empty, cp, cw, lane);
    }
  }
}

}  // namespace

// per-device one-time opt-in to the kernel's dynamic shared memory
static su2_status ensure_smem_attr() {
  static std::atomic<unsigned long long> done{0};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { set_cuda_error("cudaGetDevice", (int)e); return SU2_ERR_CUDA; }
  const unsigned long long bit = 1ull << (dev & 63);
  if (done.load(std::memory_order_acquire) & bit) return SU2_OK;
  e = cudaFuncSetAttribute(heff_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_DOUBLES_MAX * sizeof(double)));
  if (e != cudaSuccess) { set_cuda_error("cudaFuncSetAttribute(heff_tma_kernel)", (int)e); return SU2_ERR_CUDA; }
  done.fetch_or(bit, std::memory_order_release);
  return SU2_OK;
}

su2_status launch_heff_tma_tables(const DevWork* work, int nwork, const DevUnit* units, const DevTask* tasks, const void* maps,
                                  double* out, double* partial, int* counter, int* gangs, int num_sms, void* stream_v) {
  cudaStream_t stream = (cudaStream_t)stream_v;
  if (nwork == 0) return SU2_OK;
  su2_status st = ensure_smem_attr();
  if (st != SU2_OK) return st;
  const int grid = std::min(nwork, num_sms);
  heff_tma_kernel<<<grid, NTHREADS, SMEM_DOUBLES_MAX * sizeof(double), stream>>>(work, nwork, units, tasks, (const CUtensorMap*)maps,
                                                                               out, partial, counter, gangs);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_cuda_error("heff_tma_kernel launch", (int)e); return SU2_ERR_CUDA; }
  count_launch();
  return SU2_OK;
}

su2_status launch_heff_tma(const su2_plan* plan, double* out, double* partial, void* stream_v) {
  return launch_heff_tma_tables(plan->d_work, (int)plan->h_work.size(), plan->d_units, plan->d_tasks, plan->d_maps, out, partial,
                                plan->d_counter, plan->d_gang, plan->num_sms, stream_v);
}

}  // namespace su2
