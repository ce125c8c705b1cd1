// Tiling of the fused DMMA GEMM-pair kernel; shared by the planner (choice of tile class per
// output sector, segmentation, executed-flop count) and the kernels.
//
// A CTA (8 math warps + 4 load warps) owns a TM x TP tile of one output sector F_s and keeps it in registers as
// m8n8 DMMA accumulators: warp (wr, wc) of a WR x WC warp grid owns rows [32 wr, 32 wr + 32) and
// up to NT2 n8-tiles of columns.  Per position the first product T = A_pos[rows,:] E is formed in
// column chunks of at most NC columns (warp tile 32 x 8 NT1), scaled by coef*alpha_pos and parked
// in shared memory; the second product F_tile += T_chunk D_pos[cols, chunk]^T consumes it.
#pragma once
#include <algorithm>

namespace su2 {

constexpr int NWARPS = 8;              // consumer (math) warps: two warpgroups
constexpr int NPRODUCERS = 4;          // producer (cp.async) warps: one warpgroup; each copies a quarter of every tile
constexpr int NTHREADS = 32 * (NWARPS + NPRODUCERS);
constexpr int KS1 = 32;         // k extent of one pipeline stage of the first product (eight DMMA k4 steps)
constexpr int KS2 = 12;         // k extent of one pipeline stage of the second product (three DMMA k4 steps)
constexpr int NT1 = 3;          // n8-tiles per warp, first product
constexpr int NT2 = 9;          // n8-tiles per warp, second product
constexpr int MAX_STAGE = 8;    // upper bound of the pipeline depth (mbarrier arrays)

template <int WR>
struct TileCfg {
  static constexpr int WC = NWARPS / WR;        // warps along the columns
  static constexpr int TM = 32 * WR;            // rows of F per CTA          : 32 / 64 / 128
  static constexpr int TP = 8 * NT2 * WC;       // columns of F per CTA       : 576 / 288 / 144
  static constexpr int NC = 8 * NT1 * WC;       // max columns of a T chunk   : 192 / 96 / 48
  static constexpr int LDT = NC + 4;            // leading dimension of T in shared memory
  static constexpr int NSTAGE = (WR == 1) ? 3 : (WR == 2) ? 4 : 3;   // pipeline depth (what fits beside T in 227 KB)
  // one pipeline stage (doubles), every tile k-major [k/4][4][C+4]: A tile C = TM, E tile C = NC (KS1 deep),
  // D tile C = TP (KS2 deep).
  static constexpr int A_SZ = KS1 * (TM + 4);
  static constexpr int E_SZ = KS1 * (NC + 4);
  static constexpr int D_SZ = KS2 * (TP + 4);
  static constexpr int STAGE = (A_SZ + E_SZ > D_SZ) ? (A_SZ + E_SZ) : D_SZ;
  static constexpr int SMEM_DOUBLES = TM * LDT + NSTAGE * STAGE;
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

// DMMA issue slots of the slowest warp for ONE position of a task on ONE CTA tile (rows_valid x
// cols_valid of F, inner dims k, n), plus a per-stage overhead: the planner's cost unit.
inline double tile_pos_cost(int wr, int rows_valid, int cols_valid, int k, int n) {
  const TileShape ts = tile_shape(wr);
  const int mtmax = std::min(4, (rows_valid + 7) / 8);
  const int ntw2 = (((cols_valid + 7) / 8) + ts.wc - 1) / ts.wc;
  int nchunks, ncw_full;
  chunking(n, ts.nc, nchunks, ncw_full);
  double cost = 0.0;
  for (int c = 0; c < nchunks; ++c) {
    const int ncw = std::min(ncw_full, n - c * ncw_full);
    const int nt1w = (((ncw + 7) / 8) + ts.wc - 1) / ts.wc;
    cost += (double)mtmax * (nt1w * ((k + 3) / 4) + ntw2 * ((ncw + 3) / 4));
    cost += 4.0 * ((k + KS1 - 1) / KS1 + (ncw + KS2 - 1) / KS2);   // per-stage hand-over
  }
  return cost;
}

}  // namespace su2
