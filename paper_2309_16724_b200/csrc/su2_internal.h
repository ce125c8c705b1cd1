// Internal declarations shared by the planner (plan.cpp), the kernels (kernels.cu) and the
// Davidson driver (davidson.cu).  Not part of the C ABI (include/su2_heff.h).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "su2_heff.h"

namespace su2 {

// ---- device-side tables ---------------------------------------------------------------
// One sector task (paper Eq. (3)): F_s += coef * sum_pos alpha_pos A_pos E_s' D_pos^T.
struct DevTask {
  const double* A;        // block of the l operator applied: (m x k), or stored (k x m) if TRANS_A
  const double* D;        // block of the r operator applied: (p x n), or stored (n x p) if TRANS_D
  const double* alpha;    // device [npos] or nullptr (1.0)
  double coef;            // sector-value-table entry
  int64_t e_off;          // offset of the input sector E_s' in psi
  int32_t m, k, n, p;
  int32_t strideA, strideD;   // elements between positions (0: same block for all positions)
  int32_t npos;
  uint32_t flags;
};
enum : uint32_t { TASK_TRANS_A = 1u, TASK_TRANS_D = 2u };

// A bond whose block sectors all hold at most this many multiplets runs on heff_small_kernel (heff_small.cu)
// instead of the 128 x 144 / 64 x 288 / 32 x 576 register tiles of heff_dmma_kernel.
constexpr int SMALL_MAX_DIM = 48;

// A run of positions of one task inside one segment.
struct DevUnit {
  int32_t task, pos0, pos1, pad;
};

// One CTA-level work item: an output tile of one segment.
struct DevWork {
  int64_t dst_off;        // element offset of the sector in `out` (or of its partial copy)
  int32_t unit0, unit1;   // units [unit0, unit1)
  int32_t row0, col0;     // tile origin inside the (m x p) output block
  int32_t m, p;           // output block dims (p = leading dimension)
  int32_t to_partial;     // bit 0: dst_off refers to the partial buffer; bit 1: accumulate into dst (dst += tile)
  int32_t wr;             // tile class: warp rows WR of TileCfg<WR> (1, 2 or 4); 0 = whole sector (heff_small_kernel)
};

// Second pass of the deterministic segmented reduction: F_s = sum_{seg} partial[seg] in index order.
struct DevReduce {
  int64_t f_off, part_off, size;
  int32_t nseg;           // 0: sector receives nothing -> zero fill
  int32_t pad;
};

// Plan-time position folding: dst[e] = sum_pos alpha[pos] * src[pos * nelem + e].
struct FoldJob {
  const double* src;      // block of the family: [npos][nelem]
  int64_t dst_off;        // element offset inside the plan's folded-operator buffer
  int64_t nelem;
  int64_t alpha_off;      // offset into the plan's alpha array, -1: all ones
  int32_t npos, pad;
};

// Plan-time transposition of a right-block operator block: dst[pos][j][c] = src[pos][c][j].
struct TransposeJob {
  const double* src;      // [npos][rows][cols]
  int64_t dst_off;        // element offset inside the plan's transposed-operator buffer
  int32_t rows, cols, npos, pad;
};

// Diagonal tasks (s == s') for su2_heff_diag.
struct DevDiagTask {
  const double* A;
  const double* D;
  const double* alpha;
  double coef;
  int64_t f_off;
  int32_t m, p, strideA, strideD, npos, pad;
};

// ---- host-side plan --------------------------------------------------------------------
struct HostTask {
  int32_t out_sec, in_sec;
  int32_t fam_l, blk_l, adj_l;
  int32_t fam_r, blk_r, adj_r;
  int32_t term;
  double coef;
  int32_t m, k, n, p, npos;
};

struct PsiSector {
  int32_t il, sB, twoJ1, sC, ir, twoJ2;
  int64_t off;
  int32_t m, p;
};

}  // namespace su2

struct su2_plan {
  // problem copy (host)
  int32_t n_tot = 0, twoS_tot = 0;
  std::vector<su2_sector> sec_l, sec_r;
  std::vector<su2::PsiSector> psi;
  int64_t psi_len = 0;
  std::vector<su2::HostTask> tasks;
  // statistics
  su2_plan_info_t info{};
  bool host_only = false;
  // host images of the device tables
  std::vector<su2::DevTask> h_tasks;
  std::vector<su2::DevUnit> h_units;
  std::vector<su2::DevWork> h_work;
  std::vector<su2::DevReduce> h_reduce;
  std::vector<su2::DevDiagTask> h_diag;
  std::vector<su2::FoldJob> h_fold;    // plan-time folding jobs
  std::vector<su2::TransposeJob> h_trans;   // plan-time transposition jobs
  int64_t trans_elems = 0;
  int64_t fold_elems = 0;
  std::vector<int32_t> h_diag_begin;   // per psi sector: range into h_diag
  // device tables (owned)
  void* d_blob = nullptr;              // one allocation holding everything below
  su2::DevTask* d_tasks = nullptr;
  su2::DevUnit* d_units = nullptr;
  su2::DevWork* d_work = nullptr;
  su2::DevReduce* d_reduce = nullptr;
  su2::DevDiagTask* d_diag = nullptr;
  int32_t* d_diag_begin = nullptr;
  double* d_alpha = nullptr;
  double* d_identity = nullptr;
  double* d_fold = nullptr;            // folded operators (own allocation, freed with the plan)
  double* d_trans = nullptr;           // transposed copies of right-block families (own allocation; null if it did not fit)
  int32_t* d_counter = nullptr;
  void* d_psi_sec = nullptr;           // device copy of `psi` (PsiSector[])
  int64_t partial_elems = 0;
  int32_t num_sms = 148;
  int32_t small_dm8 = 0;               // > 0: small-block plan; largest sector dimension rounded up to 8
  int32_t small_begin[7] = {0, 0, 0, 0, 0, 0, 0};   // small plans: h_work is sorted by size class (DM8 = 8 (c + 1)); class c = [begin[c], begin[c+1])
};

namespace su2 {
// kernels.cu
su2_status launch_heff_dmma(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream);   // heff_dmma.cu
// the same kernel on caller-built tables (gemm_pair.cu); counter = zeroed device int
su2_status launch_heff_dmma_tables(const DevWork* work, int nwork, const DevUnit* units, const DevTask* tasks, const double* psi,
                                   double* out, double* partial, int* counter, int num_sms, void* stream);
su2_status launch_heff_small(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream);   // heff_small.cu
su2_status launch_apply(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream);
su2_status launch_diag(const su2_plan* plan, double* diag, void* stream);
su2_status upload_plan(su2_plan* plan, const std::vector<double>& alpha_host, const std::vector<double>& ident_host,
                       const std::vector<int64_t>& alpha_off_of_task, const std::vector<int64_t>& identA_off_of_task,
                       const std::vector<int64_t>& identD_off_of_task, const std::vector<int64_t>& foldA_off_of_task,
                       const std::vector<int64_t>& foldD_off_of_task, const std::vector<int64_t>& transD_off_of_task,
                       void* stream);
void free_plan_device(su2_plan* plan);
su2_status launch_gemm_pair(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, const double* X,
                            const double* B, double* C, void* stream);
// gemm_pair_small.cu: returns SU2_OK after launching, 1 if the item shape does not fit the small-block kernel
su2_status launch_gemm_pair_small(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, const double* X,
                                  const double* B, double* C, void* stream, int wpi_force, int nbuf_force);
void set_cuda_error(const char* what, int code);
void count_launch(int n = 1);   // kernels launched by this library since load (bench.py's gpu_launches)
// wigner (plan.cpp)
double wigner6j(int a2, int b2, int c2, int d2, int e2, int f2);
double wigner9j(int j1, int j2, int j, int k1, int k2, int k, int j1p, int j2p, int jp);
double c_hat(int j1, int j2, int j, int k1, int k2, int k, int j1p, int j2p, int jp);
}  // namespace su2
