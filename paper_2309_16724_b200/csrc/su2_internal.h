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
  int32_t ldA, ldD;           // leading dimensions of the STORED blocks
  int32_t npos;
  uint32_t flags;
  int32_t mapA, mapD, mapE;   // large-tile kernel: indices of the operands' tensor maps (su2_plan::d_maps)
  int32_t e_item;             // third coordinate of the E map (0 inside H_eff; the batch index of a GEMM-pair item)
  int32_t ldE, pad;           // leading dimension of the stored E block (n inside H_eff: Psi sectors are dense)
};
enum : uint32_t { TASK_TRANS_A = 1u, TASK_TRANS_D = 2u };

// A bond whose block sectors all hold at most this many multiplets runs on heff_small_kernel (heff_small.cu)
// instead of the 128 x 144 / 64 x 288 / 32 x 576 register tiles of heff_tma_kernel.
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
  int32_t ldo;            // leading dimension of the output block (p for Psi sectors; padded for operator blocks)
  int32_t gang;           // first slot of this item's gang in the pacing array (heff_tma.cu produce_item), -1 = none;
                          // the member index is row0 / TM, the member count floor(m / TM) (full row tiles)
};

// Second pass of the deterministic segmented reduction: F_s = sum_{seg} partial[seg] in index order.
struct DevReduce {
  int64_t f_off, part_off, size;
  int32_t nseg;           // 0: sector receives nothing -> zero fill
  int32_t pad;
};

// Plan-time position folding: dst[r][c] = sum_pos alpha[pos] * src[pos][r][c]  (dst leading dimension ld_dst).
struct FoldJob {
  const double* src;      // block of the family: [npos][rows][ld_src]
  int64_t dst_off;        // element offset inside the plan's folded-operator buffer
  int64_t alpha_off;      // offset into the plan's alpha array, -1: all ones
  int32_t rows, cols, ld_src, ld_dst;
  int32_t npos, pad;
};

// Plan-time padded copy of a block whose stored layout the bulk-tensor engine cannot read (rows not 16-byte
// aligned): dst[pos][r][c] = src[pos][r][c], leading dimension ld_src -> ld_dst.
struct CopyJob {
  const double* src;
  int64_t dst_off;        // element offset inside the plan's padded-operator buffer
  int32_t rows, cols, ld_src, ld_dst, npos, pad;
};

// One Psi sector of the padded private copy the E tiles are read from (psi_pad_kernel, every apply).
struct PsiPadJob {
  int64_t src_off, dst_off;
  int32_t rows, cols, ld_dst, pad;
};

// Where an operand block of a task lives (resolved to a device pointer by upload_plan).
struct OperandRef {
  int32_t kind;           // 0: caller's family memory, 1: plan's padded copy, 2: folded operators, 3: identity blocks
  int32_t side, fam;      // kind 0: family (side 0 = l, 1 = r)
  int64_t off;            // element offset inside that buffer
  int32_t rows, cols, ld; // STORED block: rows x cols, leading dimension ld
  int32_t npos;           // positions stored (1: the same block for every position)
};

// ---- two-pass route of the apply (heff_two_pass.cu; plan flag SU2_PLAN_TWO_PASS) --------------------------------
// A SLICE is a run of positions of one task whose intermediate T fits the plan's scratch together with the other slices
// of its GROUP (one pass-1 launch, one pass-2 launch, one reduce launch per group).
//   order 0: T_pos (m x n) = coef alpha_pos Aop_pos E,     partial[chunk] (m x p) = sum_{pos in chunk} T_pos Dop_pos^T
//   order 1: T_pos (k x p) = coef alpha_pos E Dop_pos^T,   partial[chunk] (m x p) = sum_{pos in chunk} Aop_pos T_pos
// (the cheaper of the two, which is what the paper's CC counts).  T_pos is stored row-major with pitch ldt in
// the scratch, viewed as ONE matrix of rows of ldt doubles: T_pos starts at row t_row0 + (pos - pos0) * rowsT.
struct TpSlice {
  int32_t task, pos0, npos, order;
  int32_t t_row0, ldt;
  int32_t mapA, mapD, mapE, mapT;   // tensor maps with the boxes of tp_gemm_kernel (indices into su2_plan::d_maps)
  int32_t item1, item2;             // first pass-1 / pass-2 item (CTA) of the slice inside its group
  int32_t chunk, nchunk;            // positions per pass-2 item; number of chunks (= partial slabs) of the slice
  int64_t part_off;                 // element offset of the slice's first partial slab in the workspace's two-pass area
  int32_t flags, pad;               // TP_SLICE_* (0 inside H_eff * Psi)
};
// su2_gemm_pair_batched on the same kernel (gemm_two_pass.cu): the "positions" are the batch items, each with its own E
// (third coordinate of the E map = position) and its own output C_pos = C_pos + T_pos Dop_pos^T (chunk = 1, the accumulators
// start from C_pos instead of zero, slabs are the dense m x p outputs themselves)
enum : int32_t { TP_SLICE_E_PER_POS = 1, TP_SLICE_ACCUMULATE = 2 };
struct TpGroup {                    // host only
  int32_t slice0, slice1, items1, items2, red0, red1;
  int32_t ipc1;                     // pass-1 items per CTA (consecutive items, pipeline kept full across them)
};
// F_s += sum of nslab partial slabs in index order (slabs of slab elements each, the first at part_off)
struct TpReduce {
  int64_t f_off, part_off, slab, size;
  int32_t nslab, pad;
};
constexpr int TP_TM = 64, TP_TN = 128, TP_KS = 20;   // CTA tile and k depth of a stage (heff_two_pass.cu)
constexpr int TP_LLD = TP_TM + 4, TP_RLD = TP_TN + 4; // row pitches of boxes read along the other direction

// Diagonal tasks (s == s') for su2_heff_diag.
struct DevDiagTask {
  const double* A;
  const double* D;
  const double* alpha;
  double coef;
  int64_t f_off;
  int32_t m, p, strideA, strideD, ldA, ldD, npos, pad;   // pad: index of the full task (host side)
};

// ---- host-side plan --------------------------------------------------------------------
struct HostTask {
  int32_t out_sec, in_sec;
  int32_t fam_l, blk_l, adj_l;
  int32_t fam_r, blk_r, adj_r;
  int32_t term;
  double coef;
  int32_t m, k, n, p, npos;
  int32_t wr;             // tile class of the output sector (large-tile plans)
  int32_t two_pass;       // 1: executed by the two-pass route (heff_two_pass.cu), not by the fused kernel
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
  std::vector<su2::OperandRef> h_opA, h_opD;   // per task: where its two operator blocks live
  std::vector<int64_t> h_alpha_off;            // per task: offset into the alpha array, -1: none
  std::vector<double> h_alpha, h_ident;        // alpha arrays of the rows; identity blocks (padded leading dimension)
  std::vector<const double*> fam_ptr[2];       // caller's family base pointers (device)
  std::vector<su2::DevUnit> h_units;
  std::vector<su2::DevWork> h_work;
  std::vector<su2::DevReduce> h_reduce;
  std::vector<su2::DevDiagTask> h_diag;
  std::vector<su2::FoldJob> h_fold;            // plan-time folding jobs
  std::vector<su2::CopyJob> h_copy;            // plan-time padded copies
  std::vector<su2::PsiPadJob> h_psipad;        // per Psi sector: its place in the padded private copy
  int64_t copy_elems = 0, fold_elems = 0, psipad_elems = 0;
  std::vector<int32_t> h_diag_begin;   // per psi sector: range into h_diag
  // device tables (owned)
  void* d_blob = nullptr;              // one allocation holding everything below
  su2::DevTask* d_tasks = nullptr;
  su2::DevUnit* d_units = nullptr;
  su2::DevWork* d_work = nullptr;
  su2::DevReduce* d_reduce = nullptr;
  su2::DevDiagTask* d_diag = nullptr;
  su2::PsiPadJob* d_psipad = nullptr;
  int32_t* d_diag_begin = nullptr;
  double* d_alpha = nullptr;
  double* d_identity = nullptr;
  void* d_maps = nullptr;              // CUtensorMap[] of the large-tile kernel (128 bytes each)
  int32_t nmaps = 0;
  double* d_fold = nullptr;            // folded operators (own allocation, freed with the plan)
  double* d_copy = nullptr;            // padded copies of families whose stored rows are not 16-byte aligned
  double* d_psi_pad = nullptr;         // padded private copy of Psi (E tiles are bulk-tensor loads from it)
  int32_t* d_counter = nullptr;
  int32_t* d_gang = nullptr;       // pacing slots of the large-tile kernel's gangs (reset to -1 before every launch)
  int64_t n_gang_slots = 0;
  bool gang_pacing = false;        // SU2_PLAN_GANG_PACING
  void* d_psi_sec = nullptr;           // device copy of `psi` (PsiSector[])
  int64_t partial_elems = 0;
  int32_t num_sms = 148;
  int32_t small_dm8 = 0;               // > 0: small-block plan; largest sector dimension rounded up to 8
  // two-pass route (SU2_PLAN_TWO_PASS)
  std::vector<su2::TpSlice> h_tp_slices;
  std::vector<su2::TpGroup> h_tp_groups;
  std::vector<su2::TpReduce> h_tp_reduce;
  int64_t tp_scratch_elems = 0;        // plan-owned T scratch (doubles)
  int64_t tp_partial_elems = 0;        // two-pass area of the caller's workspace, behind the fused kernel's partial tiles
  su2::TpSlice* d_tp_slices = nullptr;
  su2::TpReduce* d_tp_reduce = nullptr;
  double* d_tp_scratch = nullptr;
  bool tp_scratch_external = false;    // su2_plan_options.two_pass_scratch_dev: caller-owned, never freed here
  int32_t small_begin[7] = {0, 0, 0, 0, 0, 0, 0};   // small plans: h_work is sorted by size class (DM8 = 8 (c + 1)); class c = [begin[c], begin[c+1])
};

namespace su2 {
// heff_tma.cu: the large-tile kernel on a plan, and on caller-built tables (gemm_pair.cu; counter = zeroed device int)
su2_status launch_heff_tma(const su2_plan* plan, double* out, double* partial, void* stream);
su2_status launch_heff_tma_tables(const DevWork* work, int nwork, const DevUnit* units, const DevTask* tasks, const void* maps,
                                  double* out, double* partial, int* counter, int* gangs, int num_sms, void* stream);
// Tensor maps (tensor_maps.cpp).  box kinds of an operand block stored [npos][rows][ld] (cols valid per row):
//   cmajor: box {KSX along the columns, CT rows}  -- the block used as stored (k runs along the contiguous direction)
//   kmajor: box {CT + 4 along the columns, KSX rows} -- the block read transposed
struct MapKey {
  const void* base; int32_t rows, cols, ld, nitems; int64_t item_stride; int32_t box_c, box_r;
  bool operator<(const MapKey& o) const;
};
su2_status encode_tensor_map(void* out128, const MapKey& key);   // host; SU2_ERR_CUDA if the driver refuses
int tp_tile_rows_executed(int M);   // rows / columns the tiles of tp_gemm_kernel multiply for an M-row / N-column output
int tp_tile_cols_executed(int N);
// one launch of tp_gemm_kernel on caller-built tables (device pointers): pass 0 / 1, nitems items, ipc items per CTA
su2_status launch_tp_gemm(const TpSlice* slices, int nslices, int pass, int nitems, int ipc, const DevTask* tasks, const void* maps,
                          double* scratch, double* partial, void* stream);
su2_status launch_heff_two_pass(const su2_plan* plan, double* out, double* tp_partial, void* stream);   // heff_two_pass.cu
su2_status launch_heff_small(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream);   // heff_small.cu
su2_status launch_apply(const su2_plan* plan, const double* psi, double* out, double* partial, void* stream);
su2_status launch_diag(const su2_plan* plan, double* diag, void* stream);
su2_status upload_plan(su2_plan* plan, void* stream);
void free_plan_device(su2_plan* plan);
// route 0: automatic; 1: small-block kernel only; 2: fused large-tile kernel only; 3: FP64-FMA tile routine only
su2_status launch_gemm_pair(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, const double* X,
                            const double* B, double* C, void* stream, int route, int wpi, int nbuf);
// gemm_pair_small.cu: returns SU2_OK after launching, 1 if the item shape does not fit the small-block kernel
su2_status launch_gemm_two_pass(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, int ldA, const double* X, int ldX,
                                const double* B, int ldB, double* C, void* stream);   // gemm_two_pass.cu
su2_status gemm_scratch_alloc(void** out, size_t bytes, void* stream);   // gemm_two_pass.cu: from the library's own memory pool
su2_status launch_gemm_pair_small(int m, int k, int n, int p, int64_t batch, double alpha, const double* A, const double* X,
                                  const double* B, double* C, void* stream, int wpi_force, int nbuf_force);
void set_cuda_error(const char* what, int code);
void set_error_text(const char* what);
void count_launch(int n = 1);   // kernels launched by this library since load (bench.py's gpu_launches)
// wigner (plan.cpp)
double wigner6j(int a2, int b2, int c2, int d2, int e2, int f2);
double wigner9j(int j1, int j2, int j, int k1, int k2, int k, int j1p, int j2p, int jp);
double c_hat(int j1, int j2, int j, int k1, int k2, int k, int j1p, int j2p, int jp);
}  // namespace su2
