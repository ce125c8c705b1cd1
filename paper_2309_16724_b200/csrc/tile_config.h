// Tiling of the fused DMMA GEMM-pair kernel (heff_tma.cu); shared by the planner (choice of tile class per
// output sector, segmentation, executed-flop count) and the kernel.
//
// A CTA (12 math warps + one producer warpgroup) owns a TM x TP tile of one output sector F_s and keeps it in
// registers as m8n8 DMMA accumulators: warp (wr, wc) of a WR x WC warp grid owns rows [32 wr, 32 wr + 32) and the
// NT2 = 6 n8-tiles of columns [48 wc, 48 wc + 48).  Per position the first product T = A_pos[rows,:] E is formed
// in column chunks of at most NC columns (warp tile 32 x 16), scaled by coef*alpha_pos and parked in shared
// memory; the second product F_tile += T_chunk D_pos[cols, chunk]^T consumes it.
//
// Operand tiles are bulk-tensor (TMA) boxes, all of whose shared-memory row pitches are = 4 (mod 8) doubles so that
// every m8n8k4 fragment load is conflict-free without swizzling:
//   E (always read along its rows, "k-major"):  NEBOX boxes of KS1 rows x (48 + 4) columns
//   D k-major (block read transposed):          NDBOX boxes of KS2 rows x (144 + 4) columns
//   D c-major (block as stored):                NDBOX boxes of 144 rows x KS2 columns
//   A c-major (block as stored):                one box of TM rows x KS1 columns
//   A k-major (block read transposed):          one box of KS1 rows x (TM + 4) columns
#pragma once
#include <algorithm>

namespace su2 {

#ifndef SU2_NWARPS
#define SU2_NWARPS 12
#endif
constexpr int NWARPS = SU2_NWARPS;     // consumer (math) warps: 12 = three warpgroups, three warps per SM sub-partition
constexpr int WPB = NWARPS / 4;        // consumer warps that share one E box / one D box
constexpr int NPRODUCERS = 4;          // one producer warpgroup; a single elected thread issues every bulk-tensor copy
constexpr int NTHREADS = 32 * (NWARPS + NPRODUCERS);
constexpr int KS1 = 28;         // k extent of one pipeline stage of the first product (seven DMMA k4 steps)
constexpr int KS2 = 12;         // k extent of one pipeline stage of the second product (three DMMA k4 steps)
constexpr int NT1 = 6 / WPB;    // n8-tiles per warp, first product  (a box is 48 columns)
constexpr int NT2 = 18 / WPB;   // n8-tiles per warp, second product (a box is 144 columns)
constexpr int MAX_STAGE = 4;    // upper bound of the pipeline depth (mbarrier arrays)
constexpr int EBOX_C = 8 * NT1 * WPB, EBOX_LD = EBOX_C + 4;    // WPB warps share one E box: 48 (+4) columns
constexpr int DBOX_C = 8 * NT2 * WPB, DBOX_LD = DBOX_C + 4;    // WPB warps share one D box: 144 (+4) columns
constexpr int EBOX_SZ = KS1 * EBOX_LD;                          // doubles per E box
constexpr int DBOX_SZ = KS2 * DBOX_LD;                          // doubles per D box slot (c-major needs 144 * KS2 <= this)

template <int WR>
struct TileCfg {
  static_assert(NWARPS % (WPB * WR) == 0, "a box serves WPB warps");
  static constexpr int WC = NWARPS / WR;        // warps along the columns    : 12 / 6 / 3
  static constexpr int TM = 32 * WR;            // rows of F per CTA          : 32 / 64 / 128
  static constexpr int TP = 8 * NT2 * WC;       // columns of F per CTA       : 576 / 288 / 144
  static constexpr int NC = 8 * NT1 * WC;       // max columns of a T chunk   : 192 / 96 / 48
  static constexpr int LDT = NC + 4;            // leading dimension of T in shared memory
  static constexpr int NEBOX = WC / WPB, NDBOX = WC / WPB;
  static constexpr int NSTAGE = (WR == 1) ? 3 : 4;   // pipeline depth (what fits beside T in 227 KB)
  static constexpr int A_SZ = KS1 * (TM + 4);   // k-major A box (the larger of the two orientations)
  static constexpr int E_SZ = NEBOX * EBOX_SZ;
  static constexpr int D_SZ = NDBOX * DBOX_SZ;
  static constexpr int STAGE = (A_SZ + E_SZ > D_SZ) ? (A_SZ + E_SZ) : D_SZ;
  static constexpr int T_SZ = TM * LDT;
  static constexpr int SMEM_DOUBLES = T_SZ + NSTAGE * STAGE;
  // every box lands on a 128-byte boundary
  static_assert(A_SZ % 16 == 0 && EBOX_SZ % 16 == 0 && DBOX_SZ % 16 == 0 && T_SZ % 16 == 0 && STAGE % 16 == 0, "box alignment");
};

constexpr int SMEM_DOUBLES_MAX =
    TileCfg<1>::SMEM_DOUBLES > TileCfg<2>::SMEM_DOUBLES
        ? (TileCfg<1>::SMEM_DOUBLES > TileCfg<4>::SMEM_DOUBLES ? TileCfg<1>::SMEM_DOUBLES : TileCfg<4>::SMEM_DOUBLES)
        : (TileCfg<2>::SMEM_DOUBLES > TileCfg<4>::SMEM_DOUBLES ? TileCfg<2>::SMEM_DOUBLES : TileCfg<4>::SMEM_DOUBLES);

struct TileShape { int wr, wc, tm, tp, nc; };
inline TileShape tile_shape(int wr) { return TileShape{wr, NWARPS / wr, 32 * wr, 8 * NT2 * (NWARPS / wr), 8 * NT1 * (NWARPS / wr)}; }

// Column chunks of the intermediate T (n columns, at most nc_max per chunk, equal widths rounded to 8).
#if defined(__CUDACC__)
__host__ __device__
#endif
inline void chunking(int n, int nc_max, int& nchunks, int& ncw_full) {
  nchunks = (n + nc_max - 1) / nc_max;
  ncw_full = (((n + nchunks - 1) / nchunks) + 7) & ~7;
}

// DMMA issue slots of the slowest warp for ONE position of a task on ONE CTA tile (rows_valid x cols_valid of F,
// inner dims k, n), plus a per-stage overhead: the planner's cost unit.  Warp wc owns the fixed n8-tiles
// [NT wc, NT wc + NT) of its product, so the slowest warp is warp 0.
inline double tile_pos_cost(int wr, int rows_valid, int cols_valid, int k, int n) {
  const TileShape ts = tile_shape(wr);
  const int mtmax = std::min(4, (rows_valid + 7) / 8);
  const int nt2 = std::min(NT2, (cols_valid + 7) / 8);
  int nchunks, ncw_full;
  chunking(n, ts.nc, nchunks, ncw_full);
  double cost = 0.0;
  for (int c = 0; c < nchunks; ++c) {
    const int ncw = std::min(ncw_full, n - c * ncw_full);
    const int nt1 = std::min(NT1, (ncw + 7) / 8);
    cost += (double)mtmax * (nt1 * ((k + 3) / 4) + nt2 * ((ncw + 3) / 4));
    cost += 3.0 * ((k + KS1 - 1) / KS1 + (ncw + KS2 - 1) / KS2);   // per-stage hand-over
  }
  return cost;
}

// FP64 tensor flops the kernel really issues for one position of a task over ALL tiles of its output sector
// (m8 / n8 / k4 padding of both products; every row tile recomputes nothing: TP >= p is not required, a sector
// wider than TP forms T once per column tile).
inline double tile_pos_executed_flops(int wr, int m, int p, int k, int n) {
  const TileShape ts = tile_shape(wr);
  const double m8 = (m + 7) & ~7, p8 = (p + 7) & ~7, k4 = (k + 3) & ~3;
  const int coltiles = (p + ts.tp - 1) / ts.tp;
  int nchunks, ncw_full;
  chunking(n, ts.nc, nchunks, ncw_full);
  double f = 0.0;
  for (int c = 0; c < nchunks; ++c) {
    const int ncw = std::min(ncw_full, n - c * ncw_full);
    const double n8 = (ncw + 7) & ~7, n4 = (ncw + 3) & ~3;
    f += 2.0 * m8 * k4 * n8 * coltiles + 2.0 * m8 * n4 * p8;
  }
  return f;
}

}  // namespace su2
