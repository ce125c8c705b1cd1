// Host planner: the paper's sector-task-table and sector-value-table
// built once per bond, then sorted by output sector and cut into load-balanced segments.
// This replaces the paper's Contract Book / hash scheduling by a plan-time sort.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <tuple>

#include "su2_internal.h"
#include "tile_config.h"

namespace su2 {

// ---------------------------------------------------------------------------------------
// Wigner symbols (Appendix A, Eqs. (10)-(15)); doubled arguments.
// ---------------------------------------------------------------------------------------
// n! for n <= 170 (the largest factorial a long double holds comfortably).  The Racah sums below reach
// (sum of four spins + 1)!: validate() caps every doubled spin and rank at MAX_TWO_SPIN so that no argument
// exceeds the table and the alternating sums keep their precision (checked against exact rational arithmetic in
// tests/test_planner_cpu.py up to that cap).
constexpr int MAX_TWO_SPIN = 40;            // S, k <= 20
struct FactorialTable {
  long double v[171];
  FactorialTable() {
    v[0] = 1.0L;
    for (int i = 1; i <= 170; ++i) v[i] = v[i - 1] * i;
  }
};
static const long double* factorial_table() {
  static const FactorialTable tab;          // function-local static: initialised once, thread-safe
  return tab.v;
}
static inline long double fact2(int two_x) { return factorial_table()[two_x / 2]; }  // (two_x/2)!
static inline bool triad(int a, int b, int c) { return ((a + b + c) % 2 == 0) && std::abs(a - b) <= c && c <= a + b; }
// g~(a,b,c)^2 of Eq. (15)
static inline long double gsq(int a, int b, int c) {
  return fact2(a + b - c) * fact2(a - b + c) * fact2(-a + b + c) / fact2(a + b + c + 2);
}

// Eq. (13)-(14).
double wigner6j(int a, int b, int c, int d, int e, int f) {
  if (!(triad(a, b, c) && triad(c, d, e) && triad(a, e, f) && triad(b, d, f))) return 0.0;
  const int n2 = a + b + c, n3 = c + d + e, n4 = a + e + f, n5 = b + d + f;
  const int n6 = a + b + d + e, n7 = a + c + d + f, n8 = b + c + e + f;
  const int nmin = std::max(std::max(n2, n3), std::max(n4, n5));
  const int nmax = std::min(n6, std::min(n7, n8));
  long double s = 0.0L;
  for (int n = nmin; n <= nmax; n += 2) {
    long double term = fact2(n + 2) / (fact2(n - n2) * fact2(n - n3) * fact2(n - n4) * fact2(n - n5) *
                                       fact2(n6 - n) * fact2(n7 - n) * fact2(n8 - n));
    s += ((n / 2) % 2) ? -term : term;
  }
  return (double)(s * sqrtl(gsq(a, b, c) * gsq(c, d, e) * gsq(a, e, f) * gsq(b, d, f)));
}

// Eq. (10)-(12), PAPER.md:351-367 (x_min with absolute values: DESIGN.md reading G2).
double wigner9j(int j1, int j2, int j, int k1, int k2, int k, int j1p, int j2p, int jp) {
  if (!(triad(j1, j2, j) && triad(k1, k2, k) && triad(j1p, j2p, jp) && triad(j1, k1, j1p) && triad(j2, k2, j2p) &&
        triad(j, k, jp)))
    return 0.0;
  const int xmin = std::max(std::abs(j1 - jp), std::max(std::abs(j2 - k), std::abs(k1 - j2p)));
  const int xmax = std::min(j1 + jp, std::min(j2 + k, k1 + j2p));
  double s = 0.0;
  for (int x = xmin; x <= xmax; x += 2) {
    const double sign = (x % 2) ? -1.0 : 1.0;  // (-1)^(2x)
    s += sign * (x + 1) * wigner6j(j1, j2, j, k, jp, x) * wigner6j(k1, k2, k, j2, x, j2p) *
         wigner6j(j1p, j2p, jp, x, j1, k1);
  }
  return s;
}

// SU(2) factor of Eq. (5)/(9) in the Wigner-Eckart convention of su2_heff.h:
// <(j1 j2)j||[T^k1 x U^k2]^k||(j1' j2')j'> = c_hat * <j1||T||j1'> <j2||U||j2'>.
double c_hat(int j1, int j2, int j, int k1, int k2, int k, int j1p, int j2p, int jp) {
  const double w = wigner9j(j1, j2, j, k1, k2, k, j1p, j2p, jp);
  if (w == 0.0) return 0.0;
  return std::sqrt((double)(j1 + 1) * (j2 + 1) * (jp + 1) * (k + 1)) * w;
}

static const int SITE_N[3] = {0, 1, 2};
static const int SITE_2S[3] = {0, 1, 0};

}  // namespace su2

using namespace su2;

static const int U1_SITE_N[4] = {0, 1, 1, 2};
static const int U1_SITE_M[4] = {0, 1, -1, 0};

// U(1)-only mode (su2_heff.h): sectors (N, 2Sz), operator components (dN, d2Sz), 4 x 4 site matrices.
static su2_status validate_u1(const su2_problem* p) {
  if (p->nsec_l <= 0 || p->nsec_r <= 0 || !p->sec_l || !p->sec_r || p->nsite <= 0 || !p->site_u1 || p->nterm < 0)
    return SU2_ERR_INVALID_ARGUMENT;
  if (p->nterm > 0 && !p->term) return SU2_ERR_INVALID_ARGUMENT;
  if ((p->nfam_l > 0 && !p->fam_l) || (p->nfam_r > 0 && !p->fam_r) || p->nfam_l < 0 || p->nfam_r < 0)
    return SU2_ERR_INVALID_ARGUMENT;
  for (int side = 0; side < 2; ++side) {
    const int ns = side ? p->nsec_r : p->nsec_l;
    const su2_sector* sec = side ? p->sec_r : p->sec_l;
    for (int i = 0; i < ns; ++i)
      if (sec[i].dim <= 0 || sec[i].N < 0) return SU2_ERR_INVALID_SECTOR;
    const int nf = side ? p->nfam_r : p->nfam_l;
    const su2_opfamily* fam = side ? p->fam_r : p->fam_l;
    for (int f = 0; f < nf; ++f) {
      if (fam[f].npos <= 0 || fam[f].nblk < 0) return SU2_ERR_INVALID_ARGUMENT;
      if (fam[f].nblk > 0 && (!fam[f].q_out || !fam[f].q_in || !fam[f].blk_off)) return SU2_ERR_INVALID_ARGUMENT;
      for (int b = 0; b < fam[f].nblk; ++b) {
        const int qo = fam[f].q_out[b], qi = fam[f].q_in[b];
        if (qo < 0 || qo >= ns || qi < 0 || qi >= ns) return SU2_ERR_INVALID_SECTOR;
        if (sec[qo].N != sec[qi].N + fam[f].dN || sec[qo].twoS != sec[qi].twoS + fam[f].twoK) return SU2_ERR_INVALID_SECTOR;
        if (fam[f].blk_off[b] < 0) return SU2_ERR_INVALID_ARGUMENT;
      }
    }
  }
  for (int s = 0; s < p->nsite; ++s)
    for (int o = 0; o < 4; ++o)
      for (int i = 0; i < 4; ++i) {
        const double v = p->site_u1[s].r[o][i];
        if (!std::isfinite(v)) return SU2_ERR_NOT_FINITE;
        if (v != 0.0 && (U1_SITE_N[o] != U1_SITE_N[i] + p->site_u1[s].dN || U1_SITE_M[o] != U1_SITE_M[i] + p->site_u1[s].dM))
          return SU2_ERR_INVALID_SECTOR;
      }
  for (int t = 0; t < p->nterm; ++t) {
    const su2_term& tm = p->term[t];
    if (tm.fam_l < -1 || tm.fam_l >= p->nfam_l || tm.fam_r < -1 || tm.fam_r >= p->nfam_r) return SU2_ERR_INVALID_ARGUMENT;
    if (tm.op_B < 0 || tm.op_B >= p->nsite || tm.op_C < 0 || tm.op_C >= p->nsite) return SU2_ERR_INVALID_ARGUMENT;
    if (tm.npos <= 0) return SU2_ERR_INVALID_ARGUMENT;
    const int npl = tm.fam_l >= 0 ? p->fam_l[tm.fam_l].npos : 1;
    const int npr = tm.fam_r >= 0 ? p->fam_r[tm.fam_r].npos : 1;
    if ((npl != 1 && npl != tm.npos) || (npr != 1 && npr != tm.npos)) return SU2_ERR_INVALID_ARGUMENT;
    if (tm.alpha)
      for (int i = 0; i < tm.npos; ++i)
        if (!std::isfinite(tm.alpha[i])) return SU2_ERR_NOT_FINITE;
  }
  return SU2_OK;
}

static su2_status validate(const su2_problem* p) {
  if (p && p->symmetry == SU2_SYMMETRY_U1) return validate_u1(p);
  if (p && p->symmetry != SU2_SYMMETRY_SU2) return SU2_ERR_INVALID_ARGUMENT;
  if (p && (p->twoS_tot < 0 || p->twoS_tot > MAX_TWO_SPIN)) return SU2_ERR_INVALID_RANK;
  if (!p || p->nsec_l <= 0 || p->nsec_r <= 0 || !p->sec_l || !p->sec_r || p->nsite <= 0 || !p->site || p->nterm < 0)
    return SU2_ERR_INVALID_ARGUMENT;
  if (p->nterm > 0 && !p->term) return SU2_ERR_INVALID_ARGUMENT;
  if ((p->nfam_l > 0 && !p->fam_l) || (p->nfam_r > 0 && !p->fam_r) || p->nfam_l < 0 || p->nfam_r < 0)
    return SU2_ERR_INVALID_ARGUMENT;
  for (int side = 0; side < 2; ++side) {
    const int ns = side ? p->nsec_r : p->nsec_l;
    const su2_sector* sec = side ? p->sec_r : p->sec_l;
    for (int i = 0; i < ns; ++i)
      if (sec[i].dim <= 0 || sec[i].twoS < 0 || sec[i].N < 0) return SU2_ERR_INVALID_SECTOR;
    for (int i = 0; i < ns; ++i)
      if (sec[i].twoS > MAX_TWO_SPIN) return SU2_ERR_INVALID_RANK;
    const int nf = side ? p->nfam_r : p->nfam_l;
    const su2_opfamily* fam = side ? p->fam_r : p->fam_l;
    for (int f = 0; f < nf; ++f) {
      if (fam[f].npos <= 0 || fam[f].nblk < 0 || fam[f].twoK < 0) return SU2_ERR_INVALID_ARGUMENT;
      if (fam[f].twoK > MAX_TWO_SPIN) return SU2_ERR_INVALID_RANK;
      if (fam[f].nblk > 0 && (!fam[f].q_out || !fam[f].q_in || !fam[f].blk_off)) return SU2_ERR_INVALID_ARGUMENT;
      for (int b = 0; b < fam[f].nblk; ++b) {
        const int qo = fam[f].q_out[b], qi = fam[f].q_in[b];
        if (qo < 0 || qo >= ns || qi < 0 || qi >= ns) return SU2_ERR_INVALID_SECTOR;
        if (sec[qo].N != sec[qi].N + fam[f].dN) return SU2_ERR_INVALID_SECTOR;
        if (!triad(sec[qi].twoS, fam[f].twoK, sec[qo].twoS)) return SU2_ERR_INVALID_RANK;
        if (fam[f].blk_off[b] < 0) return SU2_ERR_INVALID_ARGUMENT;
      }
    }
  }
  for (int s = 0; s < p->nsite; ++s) {
    for (int o = 0; o < 3; ++o)
      for (int i = 0; i < 3; ++i) {
        const double v = p->site[s].r[o][i];
        if (!std::isfinite(v)) return SU2_ERR_NOT_FINITE;
        if (v != 0.0 && (SITE_N[o] != SITE_N[i] + p->site[s].dN)) return SU2_ERR_INVALID_SECTOR;
        if (v != 0.0 && !triad(SITE_2S[i], p->site[s].twoK, SITE_2S[o])) return SU2_ERR_INVALID_RANK;
      }
  }
  for (int t = 0; t < p->nterm; ++t) {
    const su2_term& tm = p->term[t];
    if (tm.fam_l < -1 || tm.fam_l >= p->nfam_l || tm.fam_r < -1 || tm.fam_r >= p->nfam_r) return SU2_ERR_INVALID_ARGUMENT;
    if (tm.op_B < 0 || tm.op_B >= p->nsite || tm.op_C < 0 || tm.op_C >= p->nsite) return SU2_ERR_INVALID_ARGUMENT;
    if (tm.npos <= 0) return SU2_ERR_INVALID_ARGUMENT;
    const int kl = tm.fam_l >= 0 ? p->fam_l[tm.fam_l].twoK : 0;
    const int kr = tm.fam_r >= 0 ? p->fam_r[tm.fam_r].twoK : 0;
    const int npl = tm.fam_l >= 0 ? p->fam_l[tm.fam_l].npos : 1;
    const int npr = tm.fam_r >= 0 ? p->fam_r[tm.fam_r].npos : 1;
    if ((npl != 1 && npl != tm.npos) || (npr != 1 && npr != tm.npos)) return SU2_ERR_INVALID_ARGUMENT;
    if (tm.twoK_L != tm.twoK_R) return SU2_ERR_INVALID_RANK;  // K = 0: the Hamiltonian is a spin-zero object
    if (!triad(kl, p->site[tm.op_B].twoK, tm.twoK_L) || !triad(p->site[tm.op_C].twoK, kr, tm.twoK_R))
      return SU2_ERR_INVALID_RANK;
    if (tm.alpha)
      for (int i = 0; i < tm.npos; ++i)
        if (!std::isfinite(tm.alpha[i])) return SU2_ERR_NOT_FINITE;
  }
  return SU2_OK;
}

extern "C" su2_status su2_plan_create(su2_plan** out, const su2_problem* p, int32_t flags, void* cuda_stream) {
  return su2_plan_create_opts(out, p, flags, nullptr, cuda_stream);
}

extern "C" su2_status su2_plan_create_opts(su2_plan** out, const su2_problem* p, int32_t flags, const su2_plan_options* opts,
                                           void* cuda_stream) {
  if (!out) return SU2_ERR_INVALID_ARGUMENT;
  *out = nullptr;
  su2_status st = validate(p);
  if (st != SU2_OK) return st;
  su2_plan_options opt{};
  if (opts) opt = *opts;
  if (opt.two_pass_min_dim < 0 || opt.two_pass_scratch_bytes < 0 || opt.two_pass_chunk_k < 0) return SU2_ERR_INVALID_ARGUMENT;
  if (opt.two_pass_scratch_dev && (opt.two_pass_scratch_bytes <= 0 || ((uintptr_t)opt.two_pass_scratch_dev & 255))) return SU2_ERR_WORKSPACE;
  if (opt.two_pass_min_dim == 0) opt.two_pass_min_dim = 1;
  if (opt.two_pass_scratch_bytes == 0) opt.two_pass_scratch_bytes = (int64_t)16 << 30;
  if (opt.two_pass_chunk_k == 0) opt.two_pass_chunk_k = 4096;
  if (opt.two_pass_ipc_k < 0) return SU2_ERR_INVALID_ARGUMENT;
  if (opt.two_pass_ipc_k == 0) opt.two_pass_ipc_k = 2048;
  const auto t_start = std::chrono::steady_clock::now();

  su2_plan* plan = new su2_plan();
  plan->host_only = (flags & SU2_PLAN_HOST_ONLY) != 0;
  plan->gang_pacing = (flags & SU2_PLAN_GANG_PACING) != 0;
  plan->n_tot = p->n_tot;
  plan->twoS_tot = p->twoS_tot;
  plan->sec_l.assign(p->sec_l, p->sec_l + p->nsec_l);
  plan->sec_r.assign(p->sec_r, p->sec_r + p->nsec_r);
  const auto& sl = plan->sec_l;
  const auto& sr = plan->sec_r;

  const bool u1 = p->symmetry == SU2_SYMMETRY_U1;
  // ---- Psi sectors s = (il, sB, J1, sC, ir, J2) -----------------------------------------
  std::map<std::tuple<int, int, int, int>, std::vector<int>> by_quad;  // (il,sB,sC,ir) -> sector ids
  if (u1) {
    // U(1) mode: (il, b, 0, c, ir, 0) with particle number and 2 S_z adding up to the targets
    for (int il = 0; il < (int)sl.size(); ++il)
      for (int b = 0; b < 4; ++b)
        for (int c = 0; c < 4; ++c)
          for (int ir = 0; ir < (int)sr.size(); ++ir) {
            if (sl[il].N + U1_SITE_N[b] + U1_SITE_N[c] + sr[ir].N != p->n_tot) continue;
            if (sl[il].twoS + U1_SITE_M[b] + U1_SITE_M[c] + sr[ir].twoS != p->twoS_tot) continue;
            PsiSector s{il, b, 0, c, ir, 0, plan->psi_len, sl[il].dim, sr[ir].dim};
            by_quad[std::make_tuple(il, b, c, ir)].push_back((int)plan->psi.size());
            plan->psi.push_back(s);
            plan->psi_len += (int64_t)s.m * s.p;
          }
  }
  for (int il = 0; !u1 && il < (int)sl.size(); ++il)
    for (int sB = 0; sB < 3; ++sB)
      for (int sC = 0; sC < 3; ++sC)
        for (int ir = 0; ir < (int)sr.size(); ++ir) {
          if (sl[il].N + SITE_N[sB] + SITE_N[sC] + sr[ir].N != p->n_tot) continue;
          for (int j1 = std::abs(sl[il].twoS - SITE_2S[sB]); j1 <= sl[il].twoS + SITE_2S[sB]; j1 += 2)
            for (int j2 = std::abs(sr[ir].twoS - SITE_2S[sC]); j2 <= sr[ir].twoS + SITE_2S[sC]; j2 += 2) {
              if (!triad(j1, j2, p->twoS_tot)) continue;
              PsiSector s{il, sB, j1, sC, ir, j2, plan->psi_len, sl[il].dim, sr[ir].dim};
              by_quad[std::make_tuple(il, sB, sC, ir)].push_back((int)plan->psi.size());
              plan->psi.push_back(s);
              plan->psi_len += (int64_t)s.m * s.p;
            }
        }

  // ---- task enumeration + coefficients (sector-task-table, sector-value-table) -----------
  std::vector<double> alpha_host;                 // concatenated alpha arrays
  std::vector<int64_t> alpha_off_of_term(p->nterm, -1);
  for (int t = 0; t < p->nterm; ++t)
    if (p->term[t].alpha) {
      alpha_off_of_term[t] = (int64_t)alpha_host.size();
      alpha_host.insert(alpha_host.end(), p->term[t].alpha, p->term[t].alpha + p->term[t].npos);
    }
  std::map<std::tuple<int, int, int, int, int, int, int, int, int>, double> chat_memo;
  auto chat = [&](int a, int b, int c, int d, int e, int f, int g, int h, int i) {
    auto key = std::make_tuple(a, b, c, d, e, f, g, h, i);
    auto it = chat_memo.find(key);
    if (it != chat_memo.end()) return it->second;
    const double v = c_hat(a, b, c, d, e, f, g, h, i);
    chat_memo[key] = v;
    return v;
  };

  struct Trans { int q_in, q_out, blk; double phase; };   // applied operator: ket sector -> bra sector
  auto transitions = [&](const su2_opfamily* fam, int adj, const std::vector<su2_sector>& sec) {
    std::vector<Trans> tr;
    if (!fam) {
      for (int i = 0; i < (int)sec.size(); ++i) tr.push_back({i, i, -1, 1.0});
      return tr;
    }
    for (int b = 0; b < fam->nblk; ++b) {
      const int qo = fam->q_out[b], qi = fam->q_in[b];
      if (!adj) {
        tr.push_back({qi, qo, b, 1.0});
      } else {
        // adjoint tensor: <j'||T~||j> = (-1)^(j-j'+k) sqrt((2j+1)/(2j'+1)) <j||T||j'>^T, T: j' -> j stored
        const int j = sec[qo].twoS, jp = sec[qi].twoS;
        const int e = (j - jp + fam->twoK) / 2;
        const double ph = ((e % 2) ? -1.0 : 1.0) * std::sqrt((double)(j + 1) / (double)(jp + 1));
        tr.push_back({qo, qi, b, ph});
      }
    }
    return tr;
  };

  // U(1) mode: coefficient = fermion sign x the two site elements (unit recoupling factor)
  for (int t = 0; u1 && t < p->nterm; ++t) {
    const su2_term& tm = p->term[t];
    const su2_opfamily* fl = tm.fam_l >= 0 ? &p->fam_l[tm.fam_l] : nullptr;
    const su2_opfamily* fr = tm.fam_r >= 0 ? &p->fam_r[tm.fam_r] : nullptr;
    const su2_siteop_u1& oB = p->site_u1[tm.op_B];
    const su2_siteop_u1& oC = p->site_u1[tm.op_C];
    const int pB = oB.dN & 1, pC = oC.dN & 1, pr = fr ? (fr->dN & 1) : 0;
    auto trans_u1 = [&](const su2_opfamily* fam, int adj, const std::vector<su2_sector>& sec) {
      std::vector<Trans> tr;
      if (!fam) {
        for (int i = 0; i < (int)sec.size(); ++i) tr.push_back({i, i, -1, 1.0});
        return tr;
      }
      for (int b = 0; b < fam->nblk; ++b)
        tr.push_back(adj ? Trans{fam->q_out[b], fam->q_in[b], b, 1.0} : Trans{fam->q_in[b], fam->q_out[b], b, 1.0});
      return tr;
    };
    const auto ltr = trans_u1(fl, tm.adj_l, sl);
    const auto rtr = trans_u1(fr, tm.adj_r, sr);
    for (const Trans& lt : ltr)
      for (int bi = 0; bi < 4; ++bi)
        for (int bo = 0; bo < 4; ++bo) {
          if (oB.r[bo][bi] == 0.0) continue;
          for (int ci = 0; ci < 4; ++ci)
            for (int co = 0; co < 4; ++co) {
              if (oC.r[co][ci] == 0.0) continue;
              for (const Trans& rt : rtr) {
                auto in_it = by_quad.find(std::make_tuple(lt.q_in, bi, ci, rt.q_in));
                if (in_it == by_quad.end()) continue;
                auto out_it = by_quad.find(std::make_tuple(lt.q_out, bo, co, rt.q_out));
                if (out_it == by_quad.end()) continue;
                const int nl = sl[lt.q_in].N, nB = U1_SITE_N[bi], nC = U1_SITE_N[ci];
                const int sexp = pB * nl + pC * (nl + nB) + pr * (nl + nB + nC);
                const double coef = ((sexp % 2) ? -1.0 : 1.0) * oB.r[bo][bi] * oC.r[co][ci];
                HostTask ht;
                ht.out_sec = out_it->second[0]; ht.in_sec = in_it->second[0];
                ht.fam_l = tm.fam_l; ht.blk_l = lt.blk; ht.adj_l = fl ? tm.adj_l : 0;
                ht.fam_r = tm.fam_r; ht.blk_r = rt.blk; ht.adj_r = fr ? tm.adj_r : 0;
                ht.term = t; ht.coef = coef;
                const PsiSector& a = plan->psi[ht.out_sec];
                const PsiSector& b = plan->psi[ht.in_sec];
                ht.m = a.m; ht.k = b.m; ht.n = b.p; ht.p = a.p; ht.npos = tm.npos; ht.wr = 0;
                plan->tasks.push_back(ht);
              }
            }
        }
  }
  for (int t = 0; !u1 && t < p->nterm; ++t) {
    const su2_term& tm = p->term[t];
    const su2_opfamily* fl = tm.fam_l >= 0 ? &p->fam_l[tm.fam_l] : nullptr;
    const su2_opfamily* fr = tm.fam_r >= 0 ? &p->fam_r[tm.fam_r] : nullptr;
    const su2_siteop& oB = p->site[tm.op_B];
    const su2_siteop& oC = p->site[tm.op_C];
    const int kl = fl ? fl->twoK : 0, kr = fr ? fr->twoK : 0, kB = oB.twoK, kC = oC.twoK;
    const int k1 = tm.twoK_L, k2 = tm.twoK_R;
    const int pB = oB.dN & 1, pC = oC.dN & 1, pr = fr ? (fr->dN & 1) : 0;
    const auto ltr = transitions(fl, tm.adj_l, sl);
    const auto rtr = transitions(fr, tm.adj_r, sr);
    for (const Trans& lt : ltr)
      for (int sBi = 0; sBi < 3; ++sBi) {
        const int sBo = sBi + oB.dN;
        if (sBo < 0 || sBo > 2 || oB.r[sBo][sBi] == 0.0) continue;
        for (int sCi = 0; sCi < 3; ++sCi) {
          const int sCo = sCi + oC.dN;
          if (sCo < 0 || sCo > 2 || oC.r[sCo][sCi] == 0.0) continue;
          for (const Trans& rt : rtr) {
            auto in_it = by_quad.find(std::make_tuple(lt.q_in, sBi, sCi, rt.q_in));
            if (in_it == by_quad.end()) continue;
            auto out_it = by_quad.find(std::make_tuple(lt.q_out, sBo, sCo, rt.q_out));
            if (out_it == by_quad.end()) continue;
            // fermion sign with the KET particle numbers (operators ordered O_l O_B O_C O_r)
            const int nl = sl[lt.q_in].N, nB = SITE_N[sBi], nC = SITE_N[sCi];
            const int sexp = pB * nl + pC * (nl + nB) + pr * (nl + nB + nC);
            const double base = ((sexp % 2) ? -1.0 : 1.0) * oB.r[sBo][sBi] * oC.r[sCo][sCi] * lt.phase * rt.phase;
            const int Sl = sl[lt.q_out].twoS, Slp = sl[lt.q_in].twoS;
            const int Sr = sr[rt.q_out].twoS, Srp = sr[rt.q_in].twoS;
            for (int si : in_it->second)
              for (int so : out_it->second) {
                const PsiSector& a = plan->psi[so];
                const PsiSector& b = plan->psi[si];
                const double cl = chat(Sl, SITE_2S[sBo], a.twoJ1, kl, kB, k1, Slp, SITE_2S[sBi], b.twoJ1);
                if (cl == 0.0) continue;
                const double cr = chat(SITE_2S[sCo], Sr, a.twoJ2, kC, kr, k2, SITE_2S[sCi], Srp, b.twoJ2);
                if (cr == 0.0) continue;
                const double ct = chat(a.twoJ1, a.twoJ2, p->twoS_tot, k1, k2, 0, b.twoJ1, b.twoJ2, p->twoS_tot);
                const double coef = base * cl * cr * ct;
                if (coef == 0.0 || std::fabs(coef) < 1e-300) continue;
                HostTask ht;
                ht.out_sec = so; ht.in_sec = si;
                ht.fam_l = tm.fam_l; ht.blk_l = lt.blk; ht.adj_l = fl ? tm.adj_l : 0;
                ht.fam_r = tm.fam_r; ht.blk_r = rt.blk; ht.adj_r = fr ? tm.adj_r : 0;
                ht.term = t; ht.coef = coef;
                ht.m = a.m; ht.k = b.m; ht.n = b.p; ht.p = a.p; ht.npos = tm.npos;
                plan->tasks.push_back(ht);
              }
          }
        }
      }
  }
  // plan order: by output sector, then input sector (E reuse), then row
  std::stable_sort(plan->tasks.begin(), plan->tasks.end(), [](const HostTask& x, const HostTask& y) {
    return std::tie(x.out_sec, x.in_sec, x.term, x.blk_l, x.blk_r) < std::tie(y.out_sec, y.in_sec, y.term, y.blk_l, y.blk_r);
  });

  // ---- operand layout ---------------------------------------------------------------------
  // Leading dimension of every stored block (su2_opfamily.blk_ld; dense if absent).
  auto blk_ld = [&](int side, int f, int b) {
    const su2_opfamily& fam = side ? p->fam_r[f] : p->fam_l[f];
    const auto& sec = side ? sr : sl;
    return fam.blk_ld ? (int)fam.blk_ld[b] : (int)sec[fam.q_in[b]].dim;
  };
  for (int side = 0; side < 2; ++side) {
    const int nf = side ? p->nfam_r : p->nfam_l;
    plan->fam_ptr[side].resize(nf);
    for (int f = 0; f < nf; ++f) {
      const su2_opfamily& fam = side ? p->fam_r[f] : p->fam_l[f];
      const auto& sec = side ? sr : sl;
      plan->fam_ptr[side][f] = fam.data;
      for (int b = 0; b < fam.nblk; ++b)
        if (blk_ld(side, f, b) < sec[fam.q_in[b]].dim) { delete plan; return SU2_ERR_INVALID_ARGUMENT; }
    }
  }
  auto pad4 = [](int x) { return (x + 3) & ~3; };

  // ---- position folding (the paper's pre-contraction) -----------------------------
  // A row whose positions enter through ONE block only (the other factor is the identity or has a
  // single position) is sum_pos alpha_pos A_pos applied once: that sum does not depend on Psi, so it
  // is formed at plan time (fold_kernel) and the row's tasks become one-position tasks.
  std::vector<int> fold_side(p->nterm, -1);          // -1: not folded, 0: l family folded, 1: r family folded
  std::vector<std::vector<int64_t>> fold_blk_off(p->nterm);
  int64_t fold_elems = 0;
  for (int t = 0; t < p->nterm; ++t) {
    const su2_term& tm = p->term[t];
    const int npl = tm.fam_l >= 0 ? p->fam_l[tm.fam_l].npos : 1;
    const int npr = tm.fam_r >= 0 ? p->fam_r[tm.fam_r].npos : 1;
    if (tm.npos <= 1 || (npl > 1) == (npr > 1)) continue;
    const int side = npl > 1 ? 0 : 1;
    const int fi = side ? tm.fam_r : tm.fam_l;
    const su2_opfamily& f = side ? p->fam_r[fi] : p->fam_l[fi];
    const auto& sec = side ? sr : sl;
    fold_side[t] = side;
    fold_blk_off[t].resize(f.nblk);
    for (int b = 0; b < f.nblk; ++b) {
      fold_blk_off[t][b] = fold_elems;
      FoldJob job{};
      job.src = f.data ? f.data + f.blk_off[b] : nullptr;
      job.dst_off = fold_elems;
      job.rows = sec[f.q_out[b]].dim; job.cols = sec[f.q_in[b]].dim;
      job.ld_src = blk_ld(side, fi, b); job.ld_dst = pad4(job.cols);
      job.npos = f.npos;
      job.alpha_off = alpha_off_of_term[t];
      plan->h_fold.push_back(job);
      fold_elems += (int64_t)job.rows * job.ld_dst;
    }
  }
  plan->fold_elems = fold_elems;
  for (HostTask& ht : plan->tasks)
    if (fold_side[ht.term] >= 0) ht.npos = 1;

  // ---- small-block plan? (heff_small.cu) -------------------------------------------------------
  // Every block sector of the bond holds at most SMALL_MAX_DIM multiplets: the whole apply runs on
  // heff_small_kernel (one CTA per output sector and segment), which reads blocks of any layout with plain
  // cp.async.  SU2_PLAN_LARGE_TILES keeps the large-tile kernel (tests, A/B measurements).
  {
    int maxdim = 0;
    for (const su2_sector& q : plan->sec_l) maxdim = std::max(maxdim, (int)q.dim);
    for (const su2_sector& q : plan->sec_r) maxdim = std::max(maxdim, (int)q.dim);
    const bool off = (flags & SU2_PLAN_LARGE_TILES) != 0;
    plan->small_dm8 = (maxdim <= SMALL_MAX_DIM && !off) ? std::max(8, (maxdim + 7) & ~7) : 0;
  }
  const bool small_plan = plan->small_dm8 > 0;

  // ---- padded copies for the bulk-tensor engine ---------------------------------------------------
  // heff_tma_kernel stages every operand tile with cp.async.bulk.tensor, which needs 16-byte aligned rows.  A
  // family whose device pointer is 16-byte aligned and whose blocks all have an even offset and an even leading
  // dimension is read in place; any other family used by a non-folded row is copied once, at plan time, into a
  // plan-owned buffer with leading dimensions padded to a multiple of 4 (copy_kernel).
  std::vector<std::vector<int64_t>> copy_blk_off[2];
  copy_blk_off[0].resize(p->nfam_l);
  copy_blk_off[1].resize(p->nfam_r);
  if (!small_plan) {
    std::vector<char> used[2];
    used[0].assign(p->nfam_l, 0);
    used[1].assign(p->nfam_r, 0);
    for (const HostTask& ht : plan->tasks) {
      if (ht.fam_l >= 0 && fold_side[ht.term] != 0) used[0][ht.fam_l] = 1;
      if (ht.fam_r >= 0 && fold_side[ht.term] != 1) used[1][ht.fam_r] = 1;
    }
    int64_t off = 0;
    for (int side = 0; side < 2; ++side) {
      const int nf = side ? p->nfam_r : p->nfam_l;
      for (int f = 0; f < nf; ++f) {
        if (!used[side][f]) continue;
        const su2_opfamily& fam = side ? p->fam_r[f] : p->fam_l[f];
        const auto& sec = side ? sr : sl;
        bool aligned = ((uintptr_t)fam.data & 15) == 0;
        for (int b = 0; b < fam.nblk && aligned; ++b) aligned = !(fam.blk_off[b] & 1) && !(blk_ld(side, f, b) & 1);
        if (aligned) continue;
        copy_blk_off[side][f].resize(fam.nblk);
        for (int b = 0; b < fam.nblk; ++b) {
          copy_blk_off[side][f][b] = off;
          CopyJob job{};
          job.src = fam.data ? fam.data + fam.blk_off[b] : nullptr;
          job.dst_off = off;
          job.rows = sec[fam.q_out[b]].dim; job.cols = sec[fam.q_in[b]].dim;
          job.ld_src = blk_ld(side, f, b); job.ld_dst = pad4(job.cols); job.npos = fam.npos;
          plan->h_copy.push_back(job);
          off += (int64_t)fam.npos * job.rows * job.ld_dst;
        }
      }
    }
    plan->copy_elems = off;
    // padded private copy of Psi: the E tiles are bulk-tensor loads too
    int64_t poff = 0;
    for (const PsiSector& ps : plan->psi) {
      PsiPadJob j{};
      j.src_off = ps.off; j.dst_off = poff; j.rows = ps.m; j.cols = ps.p; j.ld_dst = pad4(ps.p);
      plan->h_psipad.push_back(j);
      poff += (int64_t)ps.m * j.ld_dst;
    }
    plan->psipad_elems = poff;
  }

  // ---- task records: where the two operator blocks of every task live ----------------------------------
  const int64_t ntask = (int64_t)plan->tasks.size();
  plan->h_tasks.resize(ntask);
  plan->h_opA.resize(ntask);
  plan->h_opD.resize(ntask);
  plan->h_alpha_off.assign(ntask, -1);
  plan->h_alpha = alpha_host;
  // identity blocks: one (dim x pad4(dim)) identity per distinct dim, concatenated
  std::map<int, int64_t> ident_off;
  auto ident_for = [&](int dim) {
    auto it = ident_off.find(dim);
    if (it != ident_off.end()) return it->second;
    const int ld = pad4(dim);
    const int64_t off = (int64_t)plan->h_ident.size();
    plan->h_ident.resize(off + (int64_t)dim * ld, 0.0);
    for (int i = 0; i < dim; ++i) plan->h_ident[off + (int64_t)i * ld + i] = 1.0;
    ident_off[dim] = off;
    return off;
  };
  auto operand = [&](int side, int fam, int blk, int term, int dim) {
    OperandRef r{};
    const auto& sec = side ? sr : sl;
    if (fam < 0) {
      r.kind = 3; r.off = ident_for(dim); r.rows = dim; r.cols = dim; r.ld = pad4(dim); r.npos = 1;
      return r;
    }
    const su2_opfamily& f = side ? p->fam_r[fam] : p->fam_l[fam];
    r.side = side; r.fam = fam;
    r.rows = sec[f.q_out[blk]].dim; r.cols = sec[f.q_in[blk]].dim;
    if (fold_side[term] == side) {
      r.kind = 2; r.off = fold_blk_off[term][blk]; r.ld = pad4(r.cols); r.npos = 1;
    } else if (!copy_blk_off[side][fam].empty()) {
      r.kind = 1; r.off = copy_blk_off[side][fam][blk]; r.ld = pad4(r.cols); r.npos = f.npos;
    } else {
      r.kind = 0; r.off = f.blk_off[blk]; r.ld = blk_ld(side, fam, blk); r.npos = f.npos;
    }
    return r;
  };
  double cc = 0.0, opbytes = 0.0;
  int64_t ntp = 0;
  for (int64_t i = 0; i < ntask; ++i) {
    const HostTask& ht = plan->tasks[i];
    DevTask& d = plan->h_tasks[i];
    std::memset(&d, 0, sizeof(d));
    d.coef = ht.coef;
    d.e_off = plan->psi[ht.in_sec].off;
    d.m = ht.m; d.k = ht.k; d.n = ht.n; d.p = ht.p; d.npos = ht.npos;
    d.flags = (ht.adj_l ? TASK_TRANS_A : 0u) | (ht.adj_r ? TASK_TRANS_D : 0u);
    d.mapA = d.mapD = d.mapE = -1;
    d.ldE = ht.n;
    const OperandRef ra = operand(0, ht.fam_l, ht.blk_l, ht.term, ht.m);
    const OperandRef rd = operand(1, ht.fam_r, ht.blk_r, ht.term, ht.p);
    plan->h_opA[i] = ra;
    plan->h_opD[i] = rd;
    d.ldA = ra.ld; d.ldD = rd.ld;
    d.strideA = ra.npos > 1 ? ra.rows * ra.ld : 0;
    d.strideD = rd.npos > 1 ? rd.rows * rd.ld : 0;
    const int fs = fold_side[ht.term];
    plan->h_alpha_off[i] = fs >= 0 ? -1 : alpha_off_of_term[ht.term];   // folded rows carry alpha inside the block
    const double m = ht.m, k = ht.k, n = ht.n, pp = ht.p;
    cc += ht.npos * std::min(2 * m * k * n + 2 * m * n * pp, 2 * k * n * pp + 2 * m * k * pp);
    opbytes += ht.npos * 8.0 * (m * k + n * pp);
    ntp += ht.npos;
  }

  // ---- two-pass route (heff_two_pass.cu) --------------------------------------------------------
  // The default of a large-tile plan.  Tasks whose four extents all reach two_pass_min_dim (default: every task) leave the
  // fused kernel: their intermediate T goes through a plan-owned scratch and both products run as plain GEMMs with
  // 32 x 64 register tiles per warp, two CTAs per SM.  SU2_PLAN_FUSED (or gang pacing, which is the fused kernel's) keeps
  // everything on the fused kernel.
  const bool two_pass_on = !small_plan && !(flags & (SU2_PLAN_FUSED | SU2_PLAN_GANG_PACING));
  for (HostTask& ht : plan->tasks)
    ht.two_pass = two_pass_on && std::min(std::min(ht.m, ht.k), std::min(ht.n, ht.p)) >= opt.two_pass_min_dim ? 1 : 0;

  // ---- tile class per output sector, segments, work items ---------------------------------
  // Every output sector gets the tile class (TileCfg<WR>, tile_config.h) with the lowest modelled
  // cost.  Its task list (plan order) is cut into nseg segments of equal cost; each (segment, tile)
  // is one CTA work item.  nseg == 1 writes F directly, otherwise the segments write partial
  // copies that the reduce pass sums in index order: deterministic, no atomics (row a5).
  const int nsec = (int)plan->psi.size();
  std::vector<int64_t> first_task(nsec + 1, 0);
  std::vector<int64_t> nfused(nsec, 0);           // tasks of the sector that run on the fused kernel
  for (const HostTask& ht : plan->tasks) {
    first_task[ht.out_sec + 1]++;
    if (!ht.two_pass) nfused[ht.out_sec]++;
  }
  for (int s = 0; s < nsec; ++s) first_task[s + 1] += first_task[s];
  // cost of one position of task ht summed over all tiles of its output sector
  auto pos_cost_all_tiles = [&](int wr, const HostTask& ht) {
    const TileShape ts = tile_shape(wr);
    double c = 0.0;
    for (int r0 = 0; r0 < ht.m; r0 += ts.tm)
      for (int c0 = 0; c0 < ht.p; c0 += ts.tp)
        c += tile_pos_cost(wr, std::min(ts.tm, ht.m - r0), std::min(ts.tp, ht.p - c0), ht.k, ht.n);
    return c;
  };
  std::vector<int> sec_wr(nsec, 1);
  std::vector<double> sec_cost(nsec, 0.0);        // summed over tiles
  double total_cost = 0.0;
  for (int s = 0; s < nsec; ++s) {
    if (nfused[s] == 0) continue;
    double best = -1.0;
    for (int wr : {1, 2, 4}) {
      if (small_plan && wr != 4) continue;   // cost unit of a small plan: the 128 x 144 class (one tile per sector)
      double c = 0.0;
      for (int64_t i = first_task[s]; i < first_task[s + 1]; ++i)
        if (!plan->tasks[i].two_pass) c += pos_cost_all_tiles(wr, plan->tasks[i]) * plan->tasks[i].npos;
      if (best < 0.0 || c < best * 0.97) {   // prefer the smaller tile unless the larger one is clearly cheaper
        if (best < 0.0 || c < best) { best = c; sec_wr[s] = wr; }
      }
    }
    if (small_plan)   // + the fixed cost of a step (see step_cost below)
      for (int64_t i = first_task[s]; i < first_task[s + 1]; ++i) best += 60.0 * plan->tasks[i].npos;
    sec_cost[s] = best;
    total_cost += best;
  }
  for (HostTask& ht : plan->tasks) ht.wr = sec_wr[ht.out_sec];
  // FP64 tensor flops the kernels issue per apply (m8 / n8 / k4 padding of both products; the first product is
  // always A E, and a sector wider than its tile class forms T once per column tile); agrees with ncu's
  // sm__ops_path_tensor_src_fp64 up to the DMMAs of the predicated ragged-edge code paths
  double executed = 0.0;
  for (const HostTask& ht : plan->tasks) {
    if (ht.two_pass) {   // tp_gemm_kernel: 64 x 128 tiles with narrower ragged tiles, k padded to 4, the cheaper order
      const bool o1 = 2.0 * ht.m * ht.k * ht.n + 2.0 * ht.m * ht.n * ht.p > 2.0 * ht.k * ht.n * ht.p + 2.0 * ht.m * ht.k * ht.p;
      const double M1 = o1 ? ht.k : ht.m, N1 = o1 ? ht.p : ht.n, K1 = o1 ? ht.n : ht.k, K2 = o1 ? ht.k : ht.n;
      auto k4 = [](double x) { return std::ceil(x / 4.0) * 4.0; };
      executed += ht.npos * 2.0 * ((double)tp_tile_rows_executed((int)M1) * tp_tile_cols_executed((int)N1) * k4(K1) +
                                   (double)tp_tile_rows_executed(ht.m) * tp_tile_cols_executed(ht.p) * k4(K2));
      continue;
    }
    if (small_plan) {   // heff_small_kernel: m8n8k4 tiles over (m8, k4, n8) and (m8, n8, p8)
      const double m8 = (ht.m + 7) & ~7, k4 = (ht.k + 3) & ~3, n8 = (ht.n + 7) & ~7, p8 = (ht.p + 7) & ~7;
      executed += ht.npos * 2.0 * (m8 * k4 * n8 + m8 * n8 * p8);
    } else {
      executed += ht.npos * tile_pos_executed_flops(ht.wr, ht.m, ht.p, ht.k, ht.n);
    }
  }
  // target cost of one work item: ~24 items per SM, but never so small that the pipeline fill dominates
  // (small plans: a step costs a few hundred cycles and up to 16 CTAs are resident per SM: ~48 items per SM, low floor)
  const double target = (flags & SU2_PLAN_FORCE_SPLIT) ? 40.0
                        : small_plan ? std::max(total_cost / (148.0 * 48.0), 3.0e2)
                                     : std::max(total_cost / (148.0 * 24.0), 2.0e4);
  plan->partial_elems = 0;
  std::vector<double> work_cost;   // for LPT ordering
  for (int s = 0; s < nsec; ++s) {
    const PsiSector& ps = plan->psi[s];
    const int64_t sz = (int64_t)ps.m * ps.p;
    const int64_t t0 = first_task[s], t1 = first_task[s + 1];
    DevReduce red{};
    red.f_off = ps.off; red.size = sz; red.part_off = 0; red.nseg = 0;
    if (nfused[s] == 0) {   // nothing from the fused kernel: zero fill (the two-pass route adds to it)
      plan->h_reduce.push_back(red);
      continue;
    }
    const int wr = sec_wr[s];
    const TileShape ts = tile_shape(wr);
    const int ntiles = ((ps.m + ts.tm - 1) / ts.tm) * ((ps.p + ts.tp - 1) / ts.tp);
    // per-tile cost of a position: the full row tile (the ragged last one is cheaper; LPT evens that out)
    // small plans: a step (one position) costs two CTA barriers and a trip to L2 whatever the block size
    const double step_cost = small_plan ? 60.0 : 0.0;
    auto pos_cost = [&](const HostTask& ht) {
      return step_cost + tile_pos_cost(wr, std::min(ts.tm, ht.m), std::min(ts.tp, ht.p), ht.k, ht.n);
    };
    double tile_work = 0.0;
    for (int64_t i = t0; i < t1; ++i)
      if (!plan->tasks[i].two_pass) tile_work += pos_cost(plan->tasks[i]) * plan->tasks[i].npos;
    int nseg = (int)std::min<double>(64.0, std::max(1.0, std::ceil(tile_work / target)));
    (void)ntiles;
    std::vector<std::pair<int32_t, int32_t>> seg_units;   // unit ranges per segment
    {
      double acc = 0.0;
      int seg = 0;
      int32_t ustart = (int32_t)plan->h_units.size();
      for (int64_t i = t0; i < t1; ++i) {
        const HostTask& ht = plan->tasks[i];
        if (ht.two_pass) continue;
        const double c = pos_cost(ht);
        int pos = 0;
        while (pos < ht.npos) {
          int take = ht.npos - pos;
          if (seg < nseg - 1) {
            const double room = tile_work * (seg + 1) / nseg - acc;
            const int fit = (int)std::floor(room / c + 1e-9);
            if (fit <= 0) {   // this segment is full: close it
              seg_units.push_back({ustart, (int32_t)plan->h_units.size()});
              ustart = (int32_t)plan->h_units.size();
              ++seg;
              continue;
            }
            take = std::min(take, fit);
          }
          plan->h_units.push_back(DevUnit{(int32_t)i, pos, pos + take, 0});
          pos += take;
          acc += c * take;
        }
      }
      seg_units.push_back({ustart, (int32_t)plan->h_units.size()});
    }
    // drop empty segments
    std::vector<std::pair<int32_t, int32_t>> segs;
    for (auto& su : seg_units)
      if (su.second > su.first) segs.push_back(su);
    nseg = (int)segs.size();
    red.nseg = nseg > 1 ? nseg : 1;
    if (nseg > 1) {
      red.part_off = plan->partial_elems;
      plan->partial_elems += (int64_t)nseg * sz;
    }
    plan->h_reduce.push_back(red);
    // Gangs (large-tile kernel, SU2_PLAN_GANG_PACING): the FULL row tiles of one (segment, column tile) read the same D_pos
    // and E boxes in the same order and get one pacing slot each (heff_tma.cu produce_item).  A ragged last row tile stays
    // outside: it has less work per position, and paced to the others it would idle its SM for the difference.
    const int nrow_full = ps.m / ts.tm;
    const int ncol = (ps.p + ts.tp - 1) / ts.tp;
    for (int g = 0; g < nseg; ++g) {
      std::vector<int32_t> gang_of(ncol, -1);
      if (plan->gang_pacing && !small_plan && nrow_full > 1)
        for (int c = 0; c < ncol; ++c) {
          gang_of[c] = (int32_t)plan->n_gang_slots;
          plan->n_gang_slots += nrow_full;
        }
      for (int r0 = 0; r0 < ps.m; r0 += ts.tm)
        for (int c0 = 0; c0 < ps.p; c0 += ts.tp) {
          double w = 0.0;
          for (int32_t u = segs[g].first; u < segs[g].second; ++u) {
            const HostTask& ht = plan->tasks[plan->h_units[u].task];
            w += (step_cost + tile_pos_cost(wr, std::min(ts.tm, ps.m - r0), std::min(ts.tp, ps.p - c0), ht.k, ht.n)) *
                 (plan->h_units[u].pos1 - plan->h_units[u].pos0);
          }
          DevWork wk{};
          wk.unit0 = segs[g].first; wk.unit1 = segs[g].second;
          wk.row0 = r0; wk.col0 = c0; wk.m = ps.m; wk.p = ps.p; wk.ldo = ps.p;
          wk.to_partial = nseg > 1 ? 1 : 0;
          wk.dst_off = nseg > 1 ? red.part_off + (int64_t)g * sz : ps.off;
          wk.wr = small_plan ? 0 : wr;
          wk.gang = (r0 + ts.tm <= ps.m) ? gang_of[c0 / ts.tp] : -1;
          plan->h_work.push_back(wk);
          work_cost.push_back(w);
        }
    }
    plan->info.nsegments += nseg;
  }
  // longest-processing-time-first order for the persistent CTAs' queue
  {
    std::vector<int64_t> order(plan->h_work.size());
    for (size_t i = 0; i < order.size(); ++i) order[i] = (int64_t)i;
    // small plans: first by size class (largest dimension over the item's tasks, rounded up to 8), see heff_small.cu
    std::vector<int> cls(order.size(), 0);
    if (small_plan) {
      for (size_t i = 0; i < order.size(); ++i) {
        int dmax = 1;
        for (int32_t u = plan->h_work[i].unit0; u < plan->h_work[i].unit1; ++u) {
          const HostTask& ht = plan->tasks[plan->h_units[u].task];
          dmax = std::max({dmax, (int)ht.m, (int)ht.k, (int)ht.n, (int)ht.p});
        }
        cls[i] = (dmax + 7) / 8 - 1;
      }
      // a class with too few items to fill the GPU joins the next larger populated class (its kernel handles any
      // smaller block; one under-filled launch less)
      {
        int count[6] = {0, 0, 0, 0, 0, 0};
        for (size_t i = 0; i < order.size(); ++i) count[cls[i]]++;
        int remap[6];
        for (int c = 0; c < 6; ++c) remap[c] = c;
        for (int c = 0; c < 5; ++c) {
          if (count[c] == 0 || count[c] >= 4 * 148) continue;
          int up = c + 1;
          while (up < 6 && count[up] == 0) ++up;
          if (up < 6) { count[up] += count[c]; count[c] = 0; remap[c] = up; }
        }
        for (int c = 0; c < 6; ++c) while (remap[remap[c]] != remap[c]) remap[c] = remap[remap[c]];
        for (size_t i = 0; i < order.size(); ++i) cls[i] = remap[cls[i]];
      }
      for (int c = 0; c < 7; ++c) plan->small_begin[c] = 0;
      for (size_t i = 0; i < order.size(); ++i) plan->small_begin[cls[i] + 1]++;
      for (int c = 0; c < 6; ++c) plan->small_begin[c + 1] += plan->small_begin[c];
    }
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) {
      if (cls[a] != cls[b]) return cls[a] < cls[b];
      return work_cost[a] > work_cost[b];
    });
    std::vector<DevWork> sorted(order.size());
    for (size_t i = 0; i < order.size(); ++i) sorted[i] = plan->h_work[order[i]];
    plan->h_work.swap(sorted);
  }

  // ---- two-pass route: slices, groups, partial slabs -----------------------------------------------------
  // Tasks in plan order (sorted by output sector).  A task's positions are cut where the scratch of the current group is
  // full; a group is one launch per pass.  Pass-2 items sum `chunk` positions each (a K loop of about two_pass_chunk_k)
  // into a partial slab; consecutive slabs of one output sector inside a group form one reduce record.
  if (two_pass_on) {
    double need = 0.0;
    int64_t min_need = 0;
    for (const HostTask& ht : plan->tasks) {
      if (!ht.two_pass) continue;
      const bool o1 = 2.0 * ht.m * ht.k * ht.n + 2.0 * ht.m * ht.n * ht.p > 2.0 * ht.k * ht.n * ht.p + 2.0 * ht.m * ht.k * ht.p;
      const int64_t per_pos = (int64_t)(o1 ? ht.k : ht.m) * pad4(o1 ? ht.p : ht.n);
      need += (double)per_pos * ht.npos + 2.0 * pad4(o1 ? ht.p : ht.n);
      min_need = std::max(min_need, per_pos + 2 * (int64_t)pad4(o1 ? ht.p : ht.n));
    }
    if (opt.two_pass_scratch_dev && opt.two_pass_scratch_bytes / 8 < min_need) {   // a caller-owned scratch cannot grow
      delete plan;
      return SU2_ERR_WORKSPACE;
    }
    int64_t cap = std::max<int64_t>(opt.two_pass_scratch_bytes / 8, min_need);
    if (need < (double)cap) cap = std::max<int64_t>((int64_t)need, min_need);
    plan->tp_scratch_elems = need > 0.0 ? cap : 0;
    if (opt.two_pass_scratch_dev && plan->tp_scratch_elems > 0) {
      plan->d_tp_scratch = (double*)opt.two_pass_scratch_dev;
      plan->tp_scratch_external = true;
    }
    int64_t cur = 0, part_cur = 0, items1 = 0, items2 = 0;
    double k1_sum = 0.0;   // inner extent of the first product summed over the pass-1 items of the group
    TpGroup grp{};
    auto close_group = [&]() {
      grp.slice1 = (int32_t)plan->h_tp_slices.size();
      grp.red1 = (int32_t)plan->h_tp_reduce.size();
      grp.items1 = (int32_t)items1; grp.items2 = (int32_t)items2;
      // pass-1 items per CTA: a K loop of about two_pass_ipc_k in total per CTA, at least ~8 waves of CTAs per launch
      {
        const double k1 = items1 > 0 ? k1_sum / (double)items1 : 1.0;
        int64_t ipc = (int64_t)std::lround((double)opt.two_pass_ipc_k / std::max(1.0, k1));
        ipc = std::min<int64_t>(ipc, items1 / (8 * 296));
        grp.ipc1 = (int32_t)std::max<int64_t>(1, std::min<int64_t>(ipc, 64));
      }
      k1_sum = 0.0;
      if (grp.slice1 > grp.slice0) plan->h_tp_groups.push_back(grp);
      plan->tp_partial_elems = std::max(plan->tp_partial_elems, part_cur);
      grp.slice0 = grp.slice1; grp.red0 = grp.red1;
      cur = 0; part_cur = 0; items1 = 0; items2 = 0;
    };
    int last_sec = -1;
    for (int64_t i = 0; i < ntask; ++i) {
      const HostTask& ht = plan->tasks[i];
      if (!ht.two_pass) continue;
      const bool o1 = 2.0 * ht.m * ht.k * ht.n + 2.0 * ht.m * ht.n * ht.p > 2.0 * ht.k * ht.n * ht.p + 2.0 * ht.m * ht.k * ht.p;
      const int rowsT = o1 ? ht.k : ht.m, colsT = o1 ? ht.p : ht.n, ldt = pad4(colsT), K2 = o1 ? ht.k : ht.n;
      const int64_t per_pos = (int64_t)rowsT * ldt;
      const int64_t tiles1 = (int64_t)((rowsT + TP_TM - 1) / TP_TM) * ((colsT + TP_TN - 1) / TP_TN);
      const int64_t tiles2 = (int64_t)((ht.m + TP_TM - 1) / TP_TM) * ((ht.p + TP_TN - 1) / TP_TN);
      const int64_t slab = ((int64_t)ht.m * ht.p + 1) & ~(int64_t)1;
      int pos = 0;
      while (pos < ht.npos) {
        int64_t start = (cur + ldt - 1) / ldt * ldt;
        int64_t fit = (plan->tp_scratch_elems - start) / per_pos;
        if (start > plan->tp_scratch_elems) fit = 0;
        // a group's launches hold at most 2^30 items and its partial area at most 2^40 elements: never reached in practice
        if (fit <= 0 || items1 > ((int64_t)1 << 30)) {
          close_group();
          last_sec = -1;
          continue;
        }
        const int take = (int)std::min<int64_t>(ht.npos - pos, fit);
        TpSlice sl{};
        sl.task = (int32_t)i; sl.pos0 = pos; sl.npos = take; sl.order = o1 ? 1 : 0;
        sl.t_row0 = (int32_t)(start / ldt); sl.ldt = ldt;
        sl.mapA = sl.mapD = sl.mapE = sl.mapT = -1;
        int chunk = std::max(1, (int)std::lround((double)opt.two_pass_chunk_k / K2));
        const int nchunk = (take + chunk - 1) / chunk;
        chunk = (take + nchunk - 1) / nchunk;
        sl.chunk = chunk; sl.nchunk = (take + chunk - 1) / chunk;
        sl.item1 = (int32_t)items1; sl.item2 = (int32_t)items2;
        sl.part_off = part_cur;
        items1 += tiles1 * take;
        k1_sum += (double)(o1 ? ht.n : ht.k) * (double)(tiles1 * take);
        items2 += tiles2 * sl.nchunk;
        if (last_sec == ht.out_sec) {
          plan->h_tp_reduce.back().nslab += sl.nchunk;
        } else {
          TpReduce r{};
          r.f_off = plan->psi[ht.out_sec].off; r.part_off = part_cur; r.slab = slab; r.size = (int64_t)ht.m * ht.p; r.nslab = sl.nchunk;
          plan->h_tp_reduce.push_back(r);
          last_sec = ht.out_sec;
        }
        part_cur += slab * sl.nchunk;
        cur = start + per_pos * take;
        pos += take;
        plan->h_tp_slices.push_back(sl);
      }
    }
    close_group();
  }

  // ---- diagonal tasks (s == s') for the preconditioner -----------------------------------
  plan->h_diag_begin.assign(nsec + 1, 0);
  for (int s = 0; s < nsec; ++s) {
    plan->h_diag_begin[s] = (int32_t)plan->h_diag.size();
    for (int64_t i = first_task[s]; i < first_task[s + 1]; ++i) {
      const HostTask& ht = plan->tasks[i];
      if (ht.in_sec != ht.out_sec) continue;
      DevDiagTask d{};
      d.A = plan->h_tasks[i].A; d.D = plan->h_tasks[i].D; d.alpha = nullptr;
      d.coef = ht.coef; d.f_off = plan->psi[s].off; d.m = ht.m; d.p = ht.p;
      d.strideA = plan->h_tasks[i].strideA; d.strideD = plan->h_tasks[i].strideD; d.npos = ht.npos;
      d.ldA = plan->h_tasks[i].ldA; d.ldD = plan->h_tasks[i].ldD;
      d.pad = (int32_t)i;   // index of the full task: upload_plan copies its patched pointers
      plan->h_diag.push_back(d);
    }
  }
  plan->h_diag_begin[nsec] = (int32_t)plan->h_diag.size();

  plan->info.psi_len = plan->psi_len;
  plan->info.ntasks = ntask;
  plan->info.ntask_positions = ntp;
  plan->info.cc_flops = cc;
  plan->info.executed_flops = executed;
  plan->info.operator_bytes = opbytes;
  // a multiple of 256: the fused kernel's partial tiles, then the two-pass route's partial slabs
  plan->info.workspace_bytes = (((plan->partial_elems * 8 + 256) + 255) & ~(int64_t)255) + ((plan->tp_partial_elems * 8 + 255) & ~(int64_t)255);
  plan->info.two_pass_tasks = 0;
  for (const HostTask& ht : plan->tasks) plan->info.two_pass_tasks += ht.two_pass;
  plan->info.two_pass_groups = (int32_t)plan->h_tp_groups.size();
  plan->info.two_pass_scratch_bytes = plan->tp_scratch_elems * 8;
  plan->info.npsi_sec = nsec;
  plan->info.nwork_items = (int64_t)plan->h_work.size();   // + the CTAs of the two-pass route's launches
  for (const TpGroup& g : plan->h_tp_groups) plan->info.nwork_items += (int64_t)g.items1 + g.items2;
  plan->info.small_plan = small_plan ? 1 : 0;
  plan->info.gang_slots = (int32_t)plan->n_gang_slots;

  if (!plan->host_only) {
    st = upload_plan(plan, cuda_stream);
    if (st != SU2_OK) {
      free_plan_device(plan);
      delete plan;
      return st;
    }
  }
  plan->info.plan_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
  *out = plan;
  return SU2_OK;
}

extern "C" su2_status su2_plan_destroy(su2_plan* plan) {
  if (!plan) return SU2_ERR_INVALID_ARGUMENT;
  free_plan_device(plan);
  delete plan;
  return SU2_OK;
}

extern "C" su2_status su2_plan_info(const su2_plan* plan, su2_plan_info_t* info) {
  if (!plan || !info) return SU2_ERR_INVALID_ARGUMENT;
  *info = plan->info;
  return SU2_OK;
}

extern "C" su2_status su2_plan_psi_layout(const su2_plan* plan, int32_t* labels, int64_t* offsets) {
  if (!plan || !labels || !offsets) return SU2_ERR_INVALID_ARGUMENT;
  for (size_t i = 0; i < plan->psi.size(); ++i) {
    const PsiSector& s = plan->psi[i];
    int32_t* l = labels + 6 * i;
    l[0] = s.il; l[1] = s.sB; l[2] = s.twoJ1; l[3] = s.sC; l[4] = s.ir; l[5] = s.twoJ2;
    offsets[i] = s.off;
  }
  offsets[plan->psi.size()] = plan->psi_len;
  return SU2_OK;
}

extern "C" su2_status su2_plan_export_tasks(const su2_plan* plan, int32_t* out_sec, int32_t* in_sec, int32_t* fam_l,
                                            int32_t* blk_l, int32_t* adj_l, int32_t* fam_r, int32_t* blk_r,
                                            int32_t* adj_r, int32_t* term, double* coef) {
  if (!plan || !out_sec || !in_sec || !fam_l || !blk_l || !adj_l || !fam_r || !blk_r || !adj_r || !term || !coef)
    return SU2_ERR_INVALID_ARGUMENT;
  for (size_t i = 0; i < plan->tasks.size(); ++i) {
    const HostTask& t = plan->tasks[i];
    out_sec[i] = t.out_sec; in_sec[i] = t.in_sec;
    fam_l[i] = t.fam_l; blk_l[i] = t.blk_l; adj_l[i] = t.adj_l;
    fam_r[i] = t.fam_r; blk_r[i] = t.blk_r; adj_r[i] = t.adj_r;
    term[i] = t.term; coef[i] = t.coef;
  }
  return SU2_OK;
}

extern "C" double su2_wigner_6j(int32_t a, int32_t b, int32_t c, int32_t d, int32_t e, int32_t f) {
  const int32_t v[6] = {a, b, c, d, e, f};
  for (int32_t x : v)
    if (x < 0 || x > MAX_TWO_SPIN) return std::nan("");
  return wigner6j(a, b, c, d, e, f);
}

extern "C" double su2_wigner_9j(int32_t j1, int32_t j2, int32_t j, int32_t k1, int32_t k2, int32_t k, int32_t j1p, int32_t j2p,
                                int32_t jp) {
  const int32_t v[9] = {j1, j2, j, k1, k2, k, j1p, j2p, jp};
  for (int32_t x : v)
    if (x < 0 || x > MAX_TWO_SPIN) return std::nan("");
  return wigner9j(j1, j2, j, k1, k2, k, j1p, j2p, jp);
}

extern "C" const char* su2_status_string(su2_status st) {
  switch (st) {
    case SU2_OK: return "ok";
    case SU2_ERR_INVALID_ARGUMENT: return "invalid argument";
    case SU2_ERR_INVALID_SECTOR: return "invalid sector reference or particle-number selection rule violated";
    case SU2_ERR_INVALID_RANK: return "operator ranks cannot be coupled (triangle rule / k1 != k2)";
    case SU2_ERR_NOT_FINITE: return "non-finite alpha or site element";
    case SU2_ERR_CUDA: return "CUDA runtime error";
    case SU2_ERR_NO_DEVICE_PLAN: return "plan has no device tables (SU2_PLAN_HOST_ONLY)";
    case SU2_ERR_WORKSPACE: return "workspace missing";
    case SU2_ERR_SCRATCH_LIMIT: return "plan needs more scratch than the library's static no-alloc array holds";
    default: return "unknown status";
  }
}

extern "C" int64_t su2_plan_export_task_views(const su2_plan* plan, su2_task_view* tasks, int64_t capacity) {
  if (!plan || plan->host_only) return -1;
  const int64_t n = (int64_t)plan->h_tasks.size();
  if (!tasks) return n;
  for (int64_t i = 0; i < std::min(n, capacity); ++i) {
    const su2::DevTask& t = plan->h_tasks[i];          // operands resolved by upload_plan
    const su2::HostTask& h = plan->tasks[i];
    su2_task_view v{};
    v.A = t.A; v.D = t.D; v.alpha = t.alpha; v.coef = t.coef;
    v.strideA = t.strideA; v.strideD = t.strideD;
    v.e_off = plan->psi[h.in_sec].off; v.f_off = plan->psi[h.out_sec].off;
    v.ldA = t.ldA; v.ldD = t.ldD;
    v.transA = (t.flags & su2::TASK_TRANS_A) ? 1 : 0; v.transD = (t.flags & su2::TASK_TRANS_D) ? 1 : 0;
    v.m = t.m; v.k = t.k; v.n = t.n; v.p = t.p; v.npos = t.npos; v.pad = 0;
    tasks[i] = v;
  }
  return n;
}
