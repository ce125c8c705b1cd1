// Renormalisation (blocking) step on the device ("5-10 % of the run time",
// PAPER.md:97 Eq. (6)-(7): the W^(l) / W^(r) use of the SU(2) factor for block x site products).
//
// The block l is enlarged by the site, l' = l + B, and an operator of the new block is carried into the new (rotated,
// truncated) basis: for every pair of new sectors (q'_out, q'_in), every position pos and every pair of channels
// c_out = (q_l, sigma) of q'_out and c_in = (q_l', sigma') of q'_in,
//
//   R'[pos][q'_out <- q'_in] += weight (-1)^(p_B N_l') <sigma||O_B||sigma'> C^(S_l, s, J | k_l, k_B, k' | S_l', s', J')
//                               * U[q'_out][rows c_out]^T  R_l[pos][q_l <- q_l']  U[q'_in][rows c_in] ,
//
// with C^ the factor of Eq. (5)/(9) in the convention of su2_heff.h (the paper's W^(l) table entry, evaluated per
// channel pair here).  Each summand is F += coef * A E D^T with A = U_out-slice^T, E = the old reduced block of that
// position, D^T = U_in-slice: EXACTLY the task of the eigensolver's hot path, so the step runs on the same two
// kernels (heff_small_kernel for blocks of at most 48 rows, heff_tma_kernel otherwise) from tables built here: one
// task per (channel pair, position) -- the position selects the E operand (third coordinate of its tensor map), the
// rotation slices are the same for all positions -- and one work item per (new block, position, tile).
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <vector>

#include "su2_internal.h"
#include "tile_config.h"

using namespace su2;

namespace {

const int RN_SITE_N[3] = {0, 1, 2};
const int RN_SITE_2S[3] = {0, 1, 0};

struct Contribution {       // one channel pair of one new block
  int cho, chi;             // channels (out, in)
  int blk_old;              // block of op_old (-1: identity)
  double coef;
};

inline size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

extern "C" su2_status su2_renormalize(const su2_blocking* bk, const su2_opfamily* op_old, const su2_siteop* op_site,
                                      int32_t twoK_new, double weight, int32_t accumulate, const su2_opfamily* op_new,
                                      void* cuda_stream) {
  if (!bk || !op_new || bk->nsec_old <= 0 || bk->nsec_new <= 0 || bk->nchan <= 0 || !bk->sec_old || !bk->sec_new || !bk->chan_new ||
      !bk->chan_old || !bk->chan_site || !bk->chan_row0 || !bk->u_off || !bk->u_ld || !bk->u || !op_new->data || twoK_new < 0 ||
      !std::isfinite(weight))
    return SU2_ERR_INVALID_ARGUMENT;
  if (op_new->nblk > 0 && (!op_new->q_out || !op_new->q_in || !op_new->blk_off)) return SU2_ERR_INVALID_ARGUMENT;
  if (op_old && (op_old->nblk < 0 || (op_old->nblk > 0 && (!op_old->q_out || !op_old->q_in || !op_old->blk_off || !op_old->data))))
    return SU2_ERR_INVALID_ARGUMENT;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const int npos = op_old ? op_old->npos : 1;
  if (npos <= 0 || op_new->npos != npos) return SU2_ERR_INVALID_ARGUMENT;
  const int kl = op_old ? op_old->twoK : 0, dNl = op_old ? op_old->dN : 0;
  const int kB = op_site ? op_site->twoK : 0, dNB = op_site ? op_site->dN : 0;
  if (op_new->dN != dNl + dNB || op_new->twoK != twoK_new || twoK_new > kl + kB || twoK_new < std::abs(kl - kB) ||
      ((kl + kB + twoK_new) & 1))
    return SU2_ERR_INVALID_RANK;

  // ---- channels per new sector ------------------------------------------------------------------------
  std::vector<std::vector<int>> chans(bk->nsec_new);
  int maxdim = 1;
  for (int c = 0; c < bk->nchan; ++c) {
    const int qn = bk->chan_new[c], ql = bk->chan_old[c], sg = bk->chan_site[c];
    if (qn < 0 || qn >= bk->nsec_new || ql < 0 || ql >= bk->nsec_old || sg < 0 || sg > 2 || bk->chan_row0[c] < 0) return SU2_ERR_INVALID_SECTOR;
    if (bk->sec_old[ql].N + RN_SITE_N[sg] != bk->sec_new[qn].N) return SU2_ERR_INVALID_SECTOR;
    chans[qn].push_back(c);
    maxdim = std::max(maxdim, (int)bk->sec_old[ql].dim);
  }
  for (int q = 0; q < bk->nsec_new; ++q) {
    if (bk->sec_new[q].dim <= 0 || (bk->u_ld[q] < bk->sec_new[q].dim)) return SU2_ERR_INVALID_SECTOR;
    maxdim = std::max(maxdim, (int)bk->sec_new[q].dim);
  }
  std::map<std::pair<int, int>, int> old_block;
  if (op_old)
    for (int b = 0; b < op_old->nblk; ++b) old_block[{op_old->q_out[b], op_old->q_in[b]}] = b;
  auto ld_old = [&](int b) { return op_old->blk_ld ? (int)op_old->blk_ld[b] : (int)bk->sec_old[op_old->q_in[b]].dim; };
  auto ld_new = [&](int b) { return op_new->blk_ld ? (int)op_new->blk_ld[b] : (int)bk->sec_new[op_new->q_in[b]].dim; };

  // ---- contributions of every new block (the paper's sector-task-table of the blocking step) -----------------
  std::vector<std::vector<Contribution>> contrib(op_new->nblk);
  for (int b = 0; b < op_new->nblk; ++b) {
    const int qo = op_new->q_out[b], qi = op_new->q_in[b];
    if (qo < 0 || qo >= bk->nsec_new || qi < 0 || qi >= bk->nsec_new) return SU2_ERR_INVALID_SECTOR;
    if (bk->sec_new[qo].N != bk->sec_new[qi].N + op_new->dN) return SU2_ERR_INVALID_SECTOR;
    const int Jo = bk->sec_new[qo].twoS, Ji = bk->sec_new[qi].twoS;
    for (int co : chans[qo])
      for (int ci : chans[qi]) {
        const int lo = bk->chan_old[co], li = bk->chan_old[ci], so = bk->chan_site[co], si = bk->chan_site[ci];
        const double rs = op_site ? op_site->r[so][si] : (so == si ? 1.0 : 0.0);
        if (rs == 0.0) continue;
        int blk = -1;
        if (op_old) {
          auto it = old_block.find({lo, li});
          if (it == old_block.end()) continue;
          blk = it->second;
        } else if (lo != li) {
          continue;
        }
        const double ch = c_hat(bk->sec_old[lo].twoS, RN_SITE_2S[so], Jo, kl, kB, twoK_new, bk->sec_old[li].twoS, RN_SITE_2S[si], Ji);
        const double sgn = ((dNB & 1) && (bk->sec_old[li].N & 1)) ? -1.0 : 1.0;
        const double coef = weight * sgn * rs * ch;
        if (coef == 0.0) continue;
        contrib[b].push_back({co, ci, blk, coef});
      }
  }

  // ---- tables ----------------------------------------------------------------------------------------------
  const bool small = maxdim <= SMALL_MAX_DIM;
  auto pad4 = [](int x) { return (x + 3) & ~3; };
  std::vector<double> h_ident;
  std::map<int, int64_t> ident_off;
  if (!op_old)
    for (int q = 0; q < bk->nsec_old; ++q) {
      const int d = bk->sec_old[q].dim;
      if (ident_off.count(d)) continue;
      ident_off[d] = (int64_t)h_ident.size();
      h_ident.resize(h_ident.size() + (size_t)d * pad4(d), 0.0);
      for (int i = 0; i < d; ++i) h_ident[ident_off[d] + (int64_t)i * pad4(d) + i] = 1.0;
    }
  std::vector<DevTask> h_tasks;
  std::vector<DevUnit> h_units;
  std::vector<DevWork> h_work;
  struct MapUse { MapKey a, d, e; };
  std::vector<MapUse> uses;       // per task (large route)
  double* out = const_cast<double*>(op_new->data);
  for (int b = 0; b < op_new->nblk; ++b) {
    const int qo = op_new->q_out[b], qi = op_new->q_in[b];
    const int Do = bk->sec_new[qo].dim, Di = bk->sec_new[qi].dim, ldo = ld_new(b);
    if (ldo < Di || op_new->blk_off[b] < 0) return SU2_ERR_INVALID_ARGUMENT;
    if (!accumulate) {
      cudaError_t e = cudaMemsetAsync(out + op_new->blk_off[b], 0, (size_t)npos * Do * ldo * sizeof(double), stream);
      if (e != cudaSuccess) { set_cuda_error("cudaMemsetAsync(new operator block)", (int)e); return SU2_ERR_CUDA; }
    }
    if (contrib[b].empty()) continue;
    // tile class of this block (large route): lowest modelled cost, like the planner
    int wr = 0;
    if (!small) {
      double best = -1.0;
      for (int cand : {1, 2, 4}) {
        const TileShape ts = tile_shape(cand);
        double c = 0.0;
        for (const Contribution& ct : contrib[b]) {
          const int k = bk->sec_old[bk->chan_old[ct.cho]].dim, n = bk->sec_old[bk->chan_old[ct.chi]].dim;
          for (int r0 = 0; r0 < Do; r0 += ts.tm)
            for (int c0 = 0; c0 < Di; c0 += ts.tp) c += tile_pos_cost(cand, std::min(ts.tm, Do - r0), std::min(ts.tp, Di - c0), k, n);
        }
        if (best < 0.0 || c < best) { best = c; wr = cand; }
      }
    }
    for (int pos = 0; pos < npos; ++pos) {
      const int32_t u0 = (int32_t)h_units.size();
      for (const Contribution& ct : contrib[b]) {
        const int lo = bk->chan_old[ct.cho], li = bk->chan_old[ct.chi];
        const int k = bk->sec_old[lo].dim, n = bk->sec_old[li].dim;
        DevTask t;
        std::memset(&t, 0, sizeof(t));
        t.A = bk->u + bk->u_off[qo] + (int64_t)bk->chan_row0[ct.cho] * bk->u_ld[qo];
        t.D = bk->u + bk->u_off[qi] + (int64_t)bk->chan_row0[ct.chi] * bk->u_ld[qi];
        t.alpha = nullptr;
        t.coef = ct.coef;
        t.m = Do; t.k = k; t.n = n; t.p = Di;
        t.strideA = 0; t.strideD = 0; t.ldA = bk->u_ld[qo]; t.ldD = bk->u_ld[qi];
        t.npos = 1; t.flags = TASK_TRANS_A | TASK_TRANS_D;
        t.mapA = t.mapD = t.mapE = -1;
        const double* ebase;
        int nitems;
        if (ct.blk_old >= 0) {
          t.ldE = ld_old(ct.blk_old);
          if (t.ldE < n) return SU2_ERR_INVALID_ARGUMENT;
          t.e_off = op_old->blk_off[ct.blk_old] + (int64_t)pos * k * t.ldE;
          t.e_item = pos;
          ebase = op_old->data + op_old->blk_off[ct.blk_old];
          nitems = npos;
        } else {
          t.ldE = pad4(k);
          t.e_off = ident_off[k];
          t.e_item = 0;
          ebase = nullptr;                 // resolved once the identity buffer has its device address
          nitems = 1;
        }
        if (!small) {
          const int tm = 32 * wr;
          MapUse mu;
          mu.a = MapKey{t.A, k, Do, t.ldA, 1, (int64_t)k * t.ldA, tm + 4, KS1};
          mu.d = MapKey{t.D, n, Di, t.ldD, 1, (int64_t)n * t.ldD, DBOX_LD, KS2};
          mu.e = MapKey{ebase, k, n, t.ldE, nitems, (int64_t)k * t.ldE, EBOX_LD, KS1};
          uses.push_back(mu);
        }
        h_units.push_back(DevUnit{(int32_t)h_tasks.size(), 0, 1, 0});
        h_tasks.push_back(t);
      }
      const int32_t u1 = (int32_t)h_units.size();
      const int tm = small ? Do : 32 * wr, tp = small ? Di : tile_shape(wr).tp;
      for (int r0 = 0; r0 < Do; r0 += tm)
        for (int c0 = 0; c0 < Di; c0 += tp) {
          DevWork w;
          std::memset(&w, 0, sizeof(w));
          w.dst_off = op_new->blk_off[b] + (int64_t)pos * Do * ldo;
          w.unit0 = u0; w.unit1 = u1; w.row0 = r0; w.col0 = c0; w.m = Do; w.p = Di; w.to_partial = 2; w.wr = small ? 0 : wr;
          w.ldo = ldo;
          h_work.push_back(w);
        }
    }
  }
  if (h_work.empty()) return SU2_OK;
  if (!small)   // items of one class next to each other: the kernel drains its pipeline when the class changes
    std::stable_sort(h_work.begin(), h_work.end(), [](const DevWork& x, const DevWork& y) { return x.wr < y.wr; });

  // ---- device image: [tensor maps][tasks][units][work][identity blocks][queue counters] ----------------------------
  const size_t b_maps = up256(small ? 0 : 3 * h_tasks.size() * 128);
  const size_t b_tasks = up256(h_tasks.size() * sizeof(DevTask)), b_units = up256(h_units.size() * sizeof(DevUnit));
  const size_t b_work = up256(h_work.size() * sizeof(DevWork)), b_ident = up256(h_ident.size() * sizeof(double));
  char* blob = nullptr;
  cudaError_t e = cudaMallocAsync((void**)&blob, b_maps + b_tasks + b_units + b_work + b_ident + 256, stream);
  if (e != cudaSuccess) { set_cuda_error("cudaMallocAsync(renormalisation tables)", (int)e); return SU2_ERR_CUDA; }
  char* d_maps = blob;
  DevTask* d_tasks = (DevTask*)(blob + b_maps);
  DevUnit* d_units = (DevUnit*)(blob + b_maps + b_tasks);
  DevWork* d_work = (DevWork*)(blob + b_maps + b_tasks + b_units);
  double* d_ident = (double*)(blob + b_maps + b_tasks + b_units + b_work);
  int* d_counter = (int*)(blob + b_maps + b_tasks + b_units + b_work + b_ident);
  su2_status st = SU2_OK;
  std::vector<unsigned char> h_maps;
  if (!small) {
    std::map<MapKey, int32_t> index;
    auto map_for = [&](MapKey key, int32_t* outi) -> su2_status {
      if (!key.base) key.base = d_ident + ident_off[key.rows];
      auto it = index.find(key);
      if (it != index.end()) { *outi = it->second; return SU2_OK; }
      const int32_t idx = (int32_t)index.size();
      h_maps.resize((size_t)(idx + 1) * 128);
      su2_status s2 = encode_tensor_map(h_maps.data() + (size_t)idx * 128, key);
      if (s2 != SU2_OK) return s2;
      index[key] = idx;
      *outi = idx;
      return SU2_OK;
    };
    for (size_t i = 0; i < h_tasks.size() && st == SU2_OK; ++i) {
      if ((st = map_for(uses[i].a, &h_tasks[i].mapA)) != SU2_OK) break;
      if ((st = map_for(uses[i].d, &h_tasks[i].mapD)) != SU2_OK) break;
      st = map_for(uses[i].e, &h_tasks[i].mapE);
    }
  }
  auto up = [&](void* dst, const void* src, size_t bytes) {
    if (st != SU2_OK || bytes == 0) return;
    cudaError_t ee = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, stream);
    if (ee != cudaSuccess) { set_cuda_error("cudaMemcpyAsync(renormalisation tables)", (int)ee); st = SU2_ERR_CUDA; }
  };
  up(d_maps, h_maps.data(), h_maps.size());
  up(d_tasks, h_tasks.data(), h_tasks.size() * sizeof(DevTask));
  up(d_units, h_units.data(), h_units.size() * sizeof(DevUnit));
  up(d_work, h_work.data(), h_work.size() * sizeof(DevWork));
  up(d_ident, h_ident.data(), h_ident.size() * sizeof(double));
  if (st == SU2_OK && cudaMemsetAsync(d_counter, 0, 64, stream) != cudaSuccess) st = SU2_ERR_CUDA;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (st == SU2_OK) {
    if (small) {
      su2_plan tmp;                                   // only the fields launch_heff_small reads
      tmp.d_work = d_work; tmp.d_units = d_units; tmp.d_tasks = d_tasks; tmp.d_counter = d_counter; tmp.num_sms = sms;
      const int cls = std::max(0, (maxdim + 7) / 8 - 1);
      for (int c = 0; c < 7; ++c) tmp.small_begin[c] = c <= cls ? 0 : (int32_t)h_work.size();
      const double* psi = op_old ? op_old->data : d_ident;
      st = launch_heff_small(&tmp, psi, out, nullptr, cuda_stream);
    } else {
      st = launch_heff_tma_tables(d_work, (int)h_work.size(), d_units, d_tasks, d_maps, out, nullptr, d_counter, nullptr, sms, cuda_stream);
    }
  }
  cudaFreeAsync(blob, stream);
  return st;
}
