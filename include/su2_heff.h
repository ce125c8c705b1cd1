/*
 * su2_heff.h -- C ABI of the B200-native SU(2) spin-adapted two-site DMRG hot path:
 * the superblock product  F = H_eff * Psi  inside a Davidson eigensolver
 * (arXiv:2309.16724; all citations are PAPER.md:<line> of the paper text).
 *
 * What the library computes.  The paper's Eq. (2)/(3),
 *
 *     F{p^F} := F{p^F} + alpha_i A_i{p^A} B_i{p^B} C_i{p^C} D_i{p^D} E{p^E},
 *
 * for models whose two site Hilbert spaces decompose into one-dimensional sectors
 * reduces per (operator-table row, sector combination, position) to
 *
 *     F_s (m x p)  +=  coef * alpha_pos * A_pos (m x k) * E_s' (k x n) * D_pos^T (n x p),
 *
 * where coef (the paper's "sector-value-table" entry) is the product of the site
 * operators' reduced elements, the fermion sign and the SU(2) factor C~ of Eq. (5)/(9)
 * for block x site, site x block and the superblock (the paper's
 * W^(l), W^(r), W^(h) look-ups), all precomputed at plan time.
 *
 * Conventions: subsystems l (left block), B (site), C (site), r (right block) in
 * Jordan-Wigner order; coupling tree ((l,B)J1,(C,r)J2)S_tot; Wigner-Eckart convention
 * <S M|T^k_q|S' M'> = <k q; S' M'|S M> <S||T||S'>; all spins are passed DOUBLED (twoS = 2S).
 * A Psi sector is s = (il, sB, twoJ1, sC, ir, twoJ2); its data is one dense row-major
 * dim_l(il) x dim_r(ir) FP64 block; Psi and F are flat vectors of these blocks in the order
 * returned by su2_plan_psi_layout.
 *
 * Ownership: the caller owns every device buffer and the CUDA stream.  Host arrays handed to
 * su2_plan_create are copied and may be freed afterwards; operator-family `data` pointers are
 * DEVICE pointers that must stay valid and unchanged while the plan is used.  The library
 * allocates on the device only what belongs to the plan (freed by su2_plan_destroy): its task tables and tensor
 * maps, the position-folded operators of one-sided rows (sum_pos alpha_pos A_pos, formed once per plan), a padded
 * copy of Psi refreshed by every apply (the large-tile kernels load their tiles with bulk-tensor copies, which need
 * 16-byte aligned rows), only for operator families whose stored layout is not 16-byte aligned, a padded copy
 * of the family (su2_plan_info_t.padded_copy_bytes; see su2_opfamily.blk_ld) and, for plans on the two-pass route
 * (SU2_PLAN_TWO_PASS, the default of large-block bonds), the scratch the intermediates T_pos go through -- unless the
 * caller hands in that buffer (su2_plan_options.two_pass_scratch_dev).
 * Errors: every entry point returns 0 on success and a negative su2_status otherwise; no
 * exceptions, no aborts, no partial state.  Results are bit-reproducible for a fixed plan.
 */
#ifndef SU2_HEFF_H
#define SU2_HEFF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int32_t su2_status;
enum {
  SU2_OK = 0,
  SU2_ERR_INVALID_ARGUMENT = -1,   /* null pointer, negative size, bad index                     */
  SU2_ERR_INVALID_SECTOR = -2,     /* block references a sector that does not exist / wrong dN  */
  SU2_ERR_INVALID_RANK = -3,       /* ranks of a row cannot be coupled (triangle rule), k1 != k2;
                                      or a doubled spin / rank above 40 (S, k <= 20: the range the
                                      factorial-based 6j/9j evaluation is validated for)          */
  SU2_ERR_NOT_FINITE = -4,         /* non-finite alpha or site element                           */
  SU2_ERR_CUDA = -5,               /* a CUDA runtime call failed (see su2_last_cuda_error)       */
  SU2_ERR_NO_DEVICE_PLAN = -6,     /* plan was created with SU2_PLAN_HOST_ONLY                   */
  SU2_ERR_WORKSPACE = -7,          /* workspace pointer null although workspace_bytes > 0        */
  SU2_ERR_SCRATCH_LIMIT = -8       /* su2_heff_apply_noalloc: the plan needs more scratch than the
                                      library's static array holds (see su2_last_cuda_error)      */
};
const char* su2_status_string(su2_status st);
const char* su2_last_cuda_error(void);
/* Number of kernels this library has launched since it was loaded (all entry points). */
int64_t su2_kernel_launch_count(void);

typedef struct su2_plan su2_plan;             /* opaque */
typedef struct su2_davidson su2_davidson;     /* opaque */

/* Block sector (N, S) with multiplicity dim = number of multiplets kept. */
typedef struct { int32_t N, twoS, dim; } su2_sector;

/* One operator *family* on a block: all position-dependent operators of one type
 * ("dense matrices of the same operator type have a third index ... labeling
 * their positions ... contiguous segments in memory").  Reduced (Wigner-Eckart) blocks. */
typedef struct {
  int32_t dN;                /* particle-number change                                          */
  int32_t twoK;              /* doubled spin rank k                                             */
  int32_t npos;              /* number of positions                                             */
  int32_t nblk;              /* number of non-zero sector blocks                                */
  const int32_t* q_out;      /* HOST [nblk]: row (bra) sector index of block b                  */
  const int32_t* q_in;       /* HOST [nblk]: column (ket) sector index of block b               */
  const int64_t* blk_off;    /* HOST [nblk]: element offset of block b inside `data`            */
  const int32_t* blk_ld;     /* HOST [nblk] or NULL: leading dimension (elements) of block b,
                                >= dim(q_in); NULL = dense (ld = dim(q_in))                    */
  const double* data;        /* DEVICE: block b = [npos][dim(q_out)][ld_b] row-major, positions
                                dim(q_out)*ld_b elements apart (pad columns are never read)    */
} su2_opfamily;
/* Layout advice (memory laid out for the TMA engine): a block whose ld_b is even, whose blk_off is even and whose
 * `data` is 16-byte aligned is read IN PLACE by the large-tile kernel (bulk tensor copies need 16-byte aligned
 * rows); ld_b a multiple of 4 keeps every row on a 32-byte sector boundary.  Any other block of a plan that runs
 * the large-tile kernel is first copied into a padded plan-owned buffer (su2_plan_info_t.plan_device_bytes grows by
 * the size of the family; su2_plan_create fails with SU2_ERR_CUDA if that does not fit). */

/* Site operator: reduced elements r[out][in] over the site multiplets 0=(N=0,S=0),
 * 1=(1,1/2), 2=(2,0) (the site basis shrinks from four to three). */
typedef struct { double r[3][3]; int32_t dN, twoK; } su2_siteop;

/* Operator-table row: the rank-0 operator
 *   X = sum_pos alpha[pos] * [[O_l x O_B]^{k1} x [O_C x O_r]^{k2}]^0,  k1 == k2.
 * The row has npos positions; a family with npos positions is indexed by pos, a family with a
 * single position (or the identity, index -1) is the same for all positions.
 * adj_l/adj_r = 1: use the adjoint tensor T~_q = (-1)^(k+q) (T_-q)^dagger of the family (its
 * stored blocks are read transposed) -- Hermitian-conjugate rows need no second copy. */
typedef struct {
  int32_t fam_l, fam_r;      /* family index on l / r, -1 = identity                            */
  int32_t op_B, op_C;        /* site operator indices                                           */
  int32_t twoK_L, twoK_R;    /* doubled ranks k1, k2                                            */
  int32_t adj_l, adj_r;
  int32_t npos;              /* positions of this row                                           */
  const double* alpha;       /* HOST [npos] or NULL (all 1.0)                                   */
} su2_term;

/* U(1)-only mode (the U(1) calculation the paper's "effective" figures are rescaled to; the
 * same tables, the same kernels, a unit recoupling factor).  Sectors are labelled by (N, 2 S_z): su2_sector.twoS holds
 * 2 S_z (may be negative), su2_opfamily.twoK the change of 2 S_z of the family's operator component, twoS_tot the target
 * 2 S_z; twoK_L / twoK_R of a row are ignored.  The site basis has its four states 0 = |0>, 1 = |up>, 2 = |down>,
 * 3 = |up down>, each a one-dimensional sector; site operators are plain 4 x 4 matrices.  The coefficient
 * of a task is the fermion sign times the two site elements; an adjoint flag reads the stored block transposed and
 * reverses (dN, d2Sz), with no phase.  A Psi sector is (il, b, 0, c, ir, 0). */
typedef struct { double r[4][4]; int32_t dN, dM; } su2_siteop_u1;
enum { SU2_SYMMETRY_SU2 = 0, SU2_SYMMETRY_U1 = 1 };

typedef struct {
  int32_t n_tot, twoS_tot;   /* target particle number and doubled total spin (U(1) mode: 2 S_z) */
  int32_t nsec_l, nsec_r;
  const su2_sector *sec_l, *sec_r;
  int32_t nfam_l, nfam_r;
  const su2_opfamily *fam_l, *fam_r;
  int32_t nsite;
  const su2_siteop* site;    /* SU(2) mode: [nsite]; U(1) mode: ignored                           */
  int32_t nterm;
  const su2_term* term;
  int32_t symmetry;          /* SU2_SYMMETRY_SU2 (0) or SU2_SYMMETRY_U1                           */
  const su2_siteop_u1* site_u1;   /* U(1) mode: [nsite]                                           */
} su2_problem;

enum {
  SU2_PLAN_DEFAULT = 0,
  SU2_PLAN_HOST_ONLY = 1,    /* no device tables: planner tests on CPU                          */
  SU2_PLAN_FORCE_SPLIT = 2,  /* tiny segments: exercises the segmented reduction on small inputs */
  SU2_PLAN_LARGE_TILES = 4,  /* keep a small-block bond on the large-tile kernel (tests, A/B measurements) */
  SU2_PLAN_GANG_PACING = 8,  /* large-tile kernel: the row tiles of an output sector, which stream the same right-block
                                operators, keep within two positions of each other, so that L2 serves them to all but
                                the first (DRAM reads -70 %, L2 hit rate 60 -> 84 % at configs[3]'s blocks); costs 2-5 %
                                of the time because a row tile on a faster SM waits -- off by default, for callers that
                                share HBM bandwidth or power with something else.  Same result bit for bit. */
  SU2_PLAN_TWO_PASS = 16,    /* (the default of every large-tile plan since round 2; accepted for clarity) the tasks run UN-FUSED,
                                the way the paper executes them (one batched GEMM per product, the position
                                sum as the inner dimension of the second): pass 1 writes
                                T_pos = coef alpha_pos A_pos E (or E D_pos^T, whichever product order is cheaper -- the order
                                the paper's CC counts) to a plan-owned scratch, pass 2 contracts it over
                                (position, inner index) into partial slabs, a fixed-order reduction adds the slabs to F_s.
                                Both passes run on 64 x 128 tiles, 32 x 64 per warp, two CTAs per SM, which the FP64 tensor
                                pipe of sm_100a rewards (0.90 of the DMMA peak at configs[3] against 0.70 for
                                the fused kernel).  Small-block plans (every sector <= 48 multiplets) are not affected.
                                Deterministic; the summation order differs from the fused kernel's, so the two agree to
                                rounding, not bit for bit. */
  SU2_PLAN_FUSED = 32        /* keep the tasks on the fused kernel (T in shared memory, no scratch): tasks with an extent
                                below su2_plan_options.two_pass_min_dim stay there anyway; with this flag all do.  For
                                callers without memory for the scratch, and for A/B measurements.  Implied by
                                SU2_PLAN_GANG_PACING. */
};

/* Tuning of SU2_PLAN_TWO_PASS (su2_plan_create_opts; 0 = default for every field). */
typedef struct {
  int32_t two_pass_min_dim;        /* a task takes the two-pass route if its four extents all reach this (default 1: all do) */
  int32_t two_pass_chunk_k;        /* target length of the inner (position, index) loop of one pass-2 CTA (default 4096)      */
  int64_t two_pass_scratch_bytes;  /* upper bound of the plan-owned scratch for T (default 16 GiB; never less than one
                                      position of the largest task; su2_plan_info_t.two_pass_scratch_bytes = what was taken) */
  int32_t two_pass_ipc_k;          /* pass 1: a CTA works through consecutive (position, tile) items until their inner
                                      extents add up to about this (default 2048; 1 = one item per CTA)                     */
  int32_t pad;
  void* two_pass_scratch_dev;      /* NULL: the plan allocates the scratch itself (freed by su2_plan_destroy).  Otherwise a
                                      DEVICE buffer of two_pass_scratch_bytes bytes (which must then be > 0), 256-byte aligned,
                                      caller-owned: it must stay valid while the plan is used, is zeroed once by
                                      su2_plan_create_opts and overwritten by every apply (two plans may share one buffer if
                                      their applies are ordered on one stream); SU2_ERR_WORKSPACE if it cannot hold one
                                      position of the largest task or is misaligned.                                         */
} su2_plan_options;

typedef struct {
  int64_t psi_len;           /* number of doubles in Psi / F                                    */
  int64_t ntasks;            /* sector tasks (paper: rows of all sector-task-tables)            */
  int64_t ntask_positions;   /* tasks counted once per position (paper's "number of tasks"); a row whose
                                positions enter through one block only is folded to ONE position   */
  double cc_flops;           /* CC = sum over task-positions of min(2mkn+2mnp, 2knp+2mkp)       */
  double executed_flops;     /* flops the kernels execute per apply (tile padding, recompute)   */
  double operator_bytes;     /* 8(mk+np) summed over task-positions (algorithmic HBM traffic)   */
  int64_t workspace_bytes;   /* device workspace su2_heff_apply needs (a multiple of 256)      */
  int32_t npsi_sec;          /* number of Psi sectors                                           */
  int32_t nsegments;         /* work segments (deterministic segmented reduction)               */
  int64_t nwork_items;       /* CTA-level work items per apply                                  */
  double plan_seconds;       /* host time spent in su2_plan_create                              */
  int64_t plan_device_bytes; /* device memory owned by the plan (tables, tensor maps, folded operators, padded copies) */
  int32_t small_plan;        /* 1: every block sector holds <= 48 multiplets, su2_heff_apply runs the small-block
                                kernel (one CTA per output sector and segment); 0: large register tiles
                                (always 0 under SU2_PLAN_LARGE_TILES) */
  int32_t gang_slots;        /* row tiles that take part in gang pacing (0 without SU2_PLAN_GANG_PACING)            */
  int64_t padded_copy_bytes; /* part of plan_device_bytes: padded copies of families that could not be read in place */
  int64_t two_pass_tasks;    /* tasks on the two-pass route (0 without SU2_PLAN_TWO_PASS)                              */
  int64_t two_pass_scratch_bytes;   /* part of plan_device_bytes: the scratch the intermediates T_pos go through       */
  int32_t two_pass_groups;   /* launch groups of the two-pass route per apply (three launches each)                    */
  int32_t pad;
} su2_plan_info_t;

/* Build the plan: enumerate the sector tasks (Eq. (3)), compute the coefficient of each
 * (sector-value-table), sort them by output sector, cut the lists into
 * load-balanced segments and upload the tables on `cuda_stream` (synchronises). */
su2_status su2_plan_create(su2_plan** out, const su2_problem* p, int32_t flags, void* cuda_stream);
/* The same with tuning options (HOST, may be NULL = defaults); negative fields: SU2_ERR_INVALID_ARGUMENT. */
su2_status su2_plan_create_opts(su2_plan** out, const su2_problem* p, int32_t flags, const su2_plan_options* opts,
                                void* cuda_stream);
su2_status su2_plan_destroy(su2_plan* plan);
su2_status su2_plan_info(const su2_plan* plan, su2_plan_info_t* info);
/* The planner's own 6j / 9j evaluation (Eqs. (10)-(15), :351-384; doubled arguments 0..40), exported so
 * that it can be checked against exact arithmetic without a GPU.  NaN for an argument out of range; 0 for
 * arguments that violate a triangle rule.  {a b c; d e f} and {j1 j2 j; k1 k2 k; j1' j2' j'}. */
double su2_wigner_6j(int32_t a, int32_t b, int32_t c, int32_t d, int32_t e, int32_t f);
double su2_wigner_9j(int32_t j1, int32_t j2, int32_t j, int32_t k1, int32_t k2, int32_t k,
                     int32_t j1p, int32_t j2p, int32_t jp);
/* labels: HOST [npsi_sec][6] = (il, sB, twoJ1, sC, ir, twoJ2); offsets: HOST [npsi_sec+1]. */
su2_status su2_plan_psi_layout(const su2_plan* plan, int32_t* labels, int64_t* offsets);

/* Host copy of the task table, for tests of the planner (HOST arrays of length ntasks):
 * out_sec/in_sec: Psi sector indices; fam/blk/adj per side (fam -1 = identity); term: the row
 * the task came from; coef: the precomputed scalar (without alpha). */
su2_status su2_plan_export_tasks(const su2_plan* plan, int32_t* out_sec, int32_t* in_sec,
                                 int32_t* fam_l, int32_t* blk_l, int32_t* adj_l,
                                 int32_t* fam_r, int32_t* blk_r, int32_t* adj_r,
                                 int32_t* term, double* coef);

/* Device view of the task table after upload (sector-task-table with resolved operands): one record per task
 * F_s += coef * sum_pos alpha[pos] * Aop_pos * E_s' * Dop_pos^T (Eq. (3)).  Aop_pos is the m x k block at
 * A + pos * strideA (row pitch ldA), or its transpose if transA (the block is then stored k x m); Dop_pos the p x n block
 * at D + pos * strideD (row pitch ldD), or stored n x p if transD; stride 0 = one block for all positions.  alpha: DEVICE
 * [npos] or NULL (all 1).  E_s' is the dense k x n block at psi + e_off, F_s the dense m x p block at out + f_off.  One-sided
 * rows appear with their operators already folded over the positions (npos = 1).  The pointers belong to the plan. */
typedef struct {
  const double* A;
  const double* D;
  const double* alpha;
  double coef;
  int64_t strideA, strideD, e_off, f_off;
  int32_t ldA, ldD, transA, transD;
  int32_t m, k, n, p, npos, pad;
} su2_task_view;
/* Writes min(capacity, ntasks) records to tasks (HOST) and returns ntasks; -1 for a NULL or host-only plan.  This is what
 * an alternative execution of the same plan needs (su2_ozaki.h: H_eff * Psi on the INT8 tensor path). */
int64_t su2_plan_export_task_views(const su2_plan* plan, su2_task_view* tasks, int64_t capacity);

/* out_dev = H_eff * psi_dev (overwrites; out must not alias psi).  Asynchronous on the stream.
 * workspace_dev: DEVICE, >= workspace_bytes, 256-byte aligned.  The workspace and the plan's work-queue counter
 * are shared by every apply of the plan: applies of ONE plan must be ordered on one stream (two plans may run
 * concurrently). */
su2_status su2_heff_apply(const su2_plan* plan, const double* psi_dev, double* out_dev,
                          void* workspace_dev, void* cuda_stream);
/* The same for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): out_dev = H_eff * psi_dev with NO workspace argument.  The partial tiles of the
 * segmented reduction live in a static device array of SU2_NOALLOC_SCRATCH_BYTES = 64 MiB inside the library (held by
 * every GPU that loads it until the process exits); the call allocates and frees nothing and is bit-identical to
 * su2_heff_apply.  A plan whose partial tiles / partial slabs exceed that size (workspace_bytes - 256 > SU2_NOALLOC_SCRATCH_BYTES;
 * BASELINE.json configs[2..3]) is rejected with SU2_ERR_SCRATCH_LIMIT and a message in su2_last_cuda_error.  The array is
 * shared by ALL calls on a device and keeps the last call's contents (no element is read before the same call wrote it,
 * so nothing needs clearing): calls that overlap on the GPU -- two streams, two plans -- race; order them on one stream.
 * psi_dev / out_dev: DEVICE, caller-owned, out must not alias psi.  Asynchronous on the stream. */
#define SU2_NOALLOC_SCRATCH_BYTES (64 * 1024 * 1024)
su2_status su2_heff_apply_noalloc(const su2_plan* plan, const double* psi_dev, double* out_dev, void* cuda_stream);
int64_t su2_noalloc_scratch_bytes(void);   /* = SU2_NOALLOC_SCRATCH_BYTES, as compiled into the library */
/* Same through HOST buffers: copies psi to the device, applies, copies the result back and
 * synchronises (the end-to-end entry point; device staging buffers inside workspace_dev, which
 * must hold workspace_bytes + 2*8*psi_len bytes). */
su2_status su2_heff_apply_host(const su2_plan* plan, const double* psi_host, double* out_host,
                               void* workspace_dev, void* cuda_stream);
/* diag_dev = diagonal of H_eff in the reduced basis (for the Davidson preconditioner). */
su2_status su2_heff_diag(const su2_plan* plan, double* diag_dev, void* cuda_stream);

/* Davidson eigensolver for the lowest eigenpair (reading G8 in DESIGN.md):
 * diagonal correction while theta < min(diag) and the Krylov direction otherwise (su2_davidson_set_preconditioner),
 * classical Gram-Schmidt applied twice, subspace <= max_subspace <= 64 (restart from the Ritz vector when full).
 * All vectors live in dav_workspace_dev (DEVICE, su2_davidson_workspace_bytes bytes, caller-owned). */
int64_t su2_davidson_workspace_bytes(const su2_plan* plan, int32_t max_subspace);
su2_status su2_davidson_create(su2_davidson** out, const su2_plan* plan, int32_t max_subspace,
                               const double* x0_dev, void* dav_workspace_dev, void* cuda_stream);
/* The same for a POSITION-SHARDED plan (one rank's share of the operator positions; all ranks hold the same Psi
 * layout and run the same Davidson algebra): `reduce` must sum vec_dev[0..n) (DEVICE) over the ranks, in place,
 * ordered on cuda_stream, and leave identical bits on every rank (an NCCL all-reduce does); it is called once for
 * the diagonal at create time and once per step on w = H_eff v, right after the local su2_heff_apply.  A non-zero
 * return aborts the call with that status.  reduce == NULL is su2_davidson_create. */
typedef int32_t (*su2_reduce_fn)(double* vec_dev, int64_t n, void* cuda_stream, void* user);   /* returns a su2_status */
su2_status su2_davidson_create_sharded(su2_davidson** out, const su2_plan* plan, int32_t max_subspace,
                                       const double* x0_dev, void* dav_workspace_dev, void* cuda_stream,
                                       su2_reduce_fn reduce, void* reduce_user);
/* One iteration: w = H_eff v (su2_heff_apply), Rayleigh-Ritz, residual, new direction (the paper gives
 * no detail, reading G8).  Everything runs on the device, ordered on cuda_stream: the k x k Ritz problem
 * is solved by one CTA, coefficients never leave device memory.  The call synchronises ONCE, at its end, for the two
 * scalars it hands back.  theta: current Ritz value; resnorm: |H x - theta x|. */
su2_status su2_davidson_step(const su2_plan* plan, su2_davidson* dav, void* workspace_dev,
                             void* cuda_stream, double* theta, double* resnorm);
/* New-direction rule.  mode 1 (default): diagonal correction t = r / (diag - theta) while theta < min(diag) (minus a
 * margin of 1e-3 of the spread of diag), else the Krylov direction t = r; mode 0: always t = r (the solver is then a
 * restarted Lanczos iteration).  Other values: SU2_ERR_INVALID_ARGUMENT. */
su2_status su2_davidson_set_preconditioner(su2_davidson* dav, int32_t mode);
su2_status su2_davidson_ritz_vector(const su2_davidson* dav, double* x_dev, void* cuda_stream);
su2_status su2_davidson_destroy(su2_davidson* dav);

/* Pre-contraction of an operator family on the device ("we form pre-contracted operators to reduce the
 * N^4 terms to N^2"): a complementary family is a linear combination over the positions of a normal
 * family of the same block with weights made of the two-electron integrals,
 *     out[b][pos'][r][c] = sum_pos W[pos'][pos] * in[b][pos][r][c]     for every sector block b,
 * i.e. per block ONE row-major GEMM (npos_out x E_b) = W (npos_out x npos_in) . IN (npos_in x E_b) with E_b = rows * ld
 * of the block (positions are contiguous per block), on FP64 tensor instructions.
 * block_elems / in_off / out_off: HOST [nblk] -- E_b and the element offsets of block b inside in_dev / out_dev (the
 * family layouts of su2_opfamily: [npos][rows][ld]); w_dev: DEVICE [npos_out][npos_in] row-major; in_dev / out_dev:
 * DEVICE, caller-owned, must not overlap.  Asynchronous on the stream, bit-reproducible.  Errors: negative sizes or
 * null pointers -> SU2_ERR_INVALID_ARGUMENT. */
su2_status su2_precontract(int32_t nblk, const int64_t* block_elems, const int64_t* in_off, const int64_t* out_off,
                           int32_t npos_in, int32_t npos_out, const double* w_dev, const double* in_dev,
                           double* out_dev, void* cuda_stream);

/* Renormalisation (blocking) step on the device (Eq. (6)-(7), :311-315): the block l
 * is enlarged by the site, l' = l + B, and the operator [O_l x O_B]^{k'} is carried into the new (rotated, truncated)
 * basis of l'.  A new sector q' = (N', J) is spanned, before the rotation, by its CHANNELS (q_l, sigma) -- block sector
 * and site multiplet coupled to J -- each contributing dim(q_l) coupled rows; U[q'] (coupled rows x D'(q'), orthonormal
 * columns) is the rotation kept by the truncation.  Per new block, position and channel pair
 *   R'[pos][q'_o <- q'_i] += weight (-1)^(p_B N_l') <sigma||O_B||sigma'> C^(S_l,s,J | k_l,k_B,k' | S_l',s',J')
 *                            U[q'_o][rows c_o]^T R_l[pos][q_l <- q_l'] U[q'_i][rows c_i]
 * (C^ = Eq. (5)/(9) in this header's convention): the same fused GEMM pair as the eigensolver's, on the same kernels. */
typedef struct {
  int32_t nsec_old; const su2_sector* sec_old;   /* HOST: sectors (N, 2S, dim) of block l                           */
  int32_t nsec_new; const su2_sector* sec_new;   /* HOST: sectors (N', 2J, D') of l' in the NEW basis               */
  int32_t nchan;                                 /* channels of all new sectors                                      */
  const int32_t* chan_new;   /* HOST [nchan]: new sector of the channel                                              */
  const int32_t* chan_old;   /* HOST [nchan]: block sector q_l                                                       */
  const int32_t* chan_site;  /* HOST [nchan]: site multiplet 0 = (0,0), 1 = (1,1/2), 2 = (2,0)                       */
  const int32_t* chan_row0;  /* HOST [nchan]: first coupled row of the channel inside U[chan_new]                    */
  const int64_t* u_off;      /* HOST [nsec_new]: element offset of U[q'] inside u                                    */
  const int32_t* u_ld;       /* HOST [nsec_new]: leading dimension of U[q'] (>= D'(q'); even, with even u_off and a
                                16-byte aligned u, for blocks of more than 48 rows: bulk-tensor copies)             */
  const double* u;           /* DEVICE: U[q'] = [coupled rows][u_ld] row-major                                       */
} su2_blocking;
/* op_old: operator family on l (NULL = identity); op_site: site operator (NULL = identity); twoK_new: rank k' of the
 * product; op_new: layout of the new family (q_out / q_in index sec_new, blk_off, blk_ld, npos = op_old's, dN and twoK
 * of the product) whose DEVICE `data` is WRITTEN (accumulate = 0: overwritten, blocks without contribution zeroed;
 * 1: added to, which is how sums of several products -- complementary operators -- are composed).  Families of more
 * than 48-row blocks must be 16-byte aligned (su2_opfamily layout advice).  Asynchronous on the stream; table memory is
 * stream-ordered.  Errors: SU2_ERR_INVALID_ARGUMENT / _SECTOR / _RANK as for su2_plan_create, SU2_ERR_CUDA. */
su2_status su2_renormalize(const su2_blocking* blocking, const su2_opfamily* op_old, const su2_siteop* op_site,
                           int32_t twoK_new, double weight, int32_t accumulate, const su2_opfamily* op_new,
                           void* cuda_stream);

/* Strided-batched FP64 GEMM-pair microbenchmark entry (BASELINE.json configs[4]):
 * C_b (m x p) += alpha * A_b (m x k) * X_b (k x n) * B_b^T (n x p) for b < batch, all DEVICE,
 * row-major, dense strides (A_b = A + b*m*k, ...); the paper's strided-batched GEMM sequences.
 * Items of at least 48 in every extent run UN-FUSED, as in the paper: T_b = alpha A_b X_b (or alpha X_b B_b^T, the cheaper
 * order) through a stream-ordered scratch, then C_b += T_b B_b^T, both on the two-pass GEMM kernel of the apply (64 x 128
 * tiles, narrower edge tiles, several consecutive tiles per CTA); an operand whose rows are not 16-byte aligned (odd k or n,
 * odd base address) is first copied into a stream-ordered buffer with an even row pitch.  Smaller items whose operands fit one
 * SM's shared memory run one CTA per item with T kept on chip (HBM-bound regime); items with one short extent use the fused
 * large-tile kernel.  C_b blocks must not overlap; one CTA owns an output element, so results are
 * bit-reproducible.  Errors: non-positive dimension, negative batch or null pointer -> SU2_ERR_INVALID_ARGUMENT; batch == 0
 * is a no-op. */
su2_status su2_gemm_pair_batched(int32_t m, int32_t k, int32_t n, int32_t p, int64_t batch, double alpha,
                                 const double* A, const double* X, const double* B, double* C,
                                 void* cuda_stream);
/* The same with the kernel chosen by the caller (tests, tuning): route 0 automatic, 1 small-block kernel, 2 fused
 * large-tile kernel, 4 un-fused two-pass kernel (T through a stream-ordered scratch; 32 x 64 register tiles per warp, two
 * CTAs per SM: chosen automatically for items of at least 48 in every extent), 3 FP64-FMA
 * tile routine (a plain reference routine, never chosen automatically below 2^24 items); SU2_ERR_INVALID_ARGUMENT if
 * the shape does not fit the route.  wpi / nbuf (0 = heuristics) override the small-block kernel's warps per item and input buffering. */
su2_status su2_gemm_pair_batched_route(int32_t m, int32_t k, int32_t n, int32_t p, int64_t batch, double alpha,
                                       const double* A, const double* X, const double* B, double* C,
                                       void* cuda_stream, int32_t route, int32_t wpi, int32_t nbuf);

#ifdef __cplusplus
}
#endif
#endif /* SU2_HEFF_H */
