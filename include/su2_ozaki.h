/*
 * su2_ozaki.h -- the strided-batched FP64 GEMM pair on the INT8 tensor path (libsu2ozaki.so).
 *
 * PAPER.md:7 and :255 quote the paper's headline against the FP64 ceiling of its GPUs.  On sm_100a the FP64 tensor
 * instruction (DMMA.8x8x4) runs at the rate of the FP64 vector pipe (37 TFLOP/s measured) and tcgen05.mma has no f64
 * kind, so the only road past that ceiling with tensor units is exact integer arithmetic: every operand is scaled by
 * powers of two per contraction line, cut into `nslices` INT8 slices of 7 bits, the slice pairs are multiplied
 * exactly on tcgen05.mma kind::i8 (int32 accumulators in TMEM) and the integer planes are recombined in FP64.  The
 * scheme is written out step by step in oracle/ozaki.py (the oracle of this entry) and DESIGN.md section 6.
 *
 * A library of its own: it is the one place where a kernel is generated from vendored header templates (the INT8 GEMM
 * comes from the CUTLASS sm_100 collective builder; slicing and recombination kernels are hand-written), and
 * libsu2heff.so does not depend on it.
 */
#ifndef SU2_OZAKI_H
#define SU2_OZAKI_H

#include <stddef.h>
#include <stdint.h>

#include "su2_heff.h"   /* su2_task_view */

#ifdef __cplusplus
extern "C" {
#endif

#define SU2_OZAKI_MAX_SLICES 7

/* C_b (m x p) += alpha * A_b (m x k) * X_b (k x n) * B_b^T (n x p) for b < batch: the operation of
 * su2_heff.h's su2_gemm_pair_batched -- PAPER.md:116-136 --, same layout (all DEVICE, row-major, dense strides
 * A_b = A + b*m*k, X_b = X + b*k*n, B_b = B + b*p*n, C_b = C + b*m*p; C_b blocks must not overlap), computed as
 * T = A X and C += alpha T B^T, each product by the sliced integer scheme above.
 *
 * nslices: 2..7 slices of 7 bits (0 = 7).  Entry-wise error of each product: <= 2^(e_i + f_j) * K * (nslices + 2) *
 * 2^(-7 nslices), e_i / f_j the binary exponents of the largest magnitude in row i of the left operand and in column
 * j of the right operand, K the contraction length (oracle/ozaki.py).  With 7 slices and N(0,1) operands the result
 * is within 1e-12 of max|C| of the FP64 product; the result is bit-reproducible (integer sums are exact, the FP64
 * recombination has a fixed order).
 *
 * Shapes are arbitrary (the INT8 copies are padded inside: contraction lengths and MN-major rows to 16 bytes, integer
 * plane rows to 4 entries, pads zero); operands 8-byte aligned (lines that start on a 16-byte boundary are read with
 * 16-byte loads).  Restriction: nslices * roundup16(max(k, n)) * 127^2 < 2^31 (exact int32 sums: k, n <= 19008 at 7
 * slices).  Inf / NaN operands are not supported (the result is unspecified).
 *
 * Memory: slices and integer planes of a chunk of items live in `workspace` (DEVICE, 256-byte aligned, workspace_bytes
 * long, owned by the caller, free for reuse once the stream has passed the call); the batch is processed in chunks of
 * as many items as fit (su2_ozaki_workspace_bytes(m, k, n, p, items, nslices) says how much `items` items need: about
 * nslices (m k + k n + m n + p n) + 4 nslices m max(n, p) bytes each, with k and n rounded up to 16 and p to 4).  workspace == NULL: a stream-ordered allocation
 * (cudaMallocAsync on cuda_stream) of at most workspace_bytes (0 = 2 GiB), freed in stream order before the call
 * returns.  Asynchronous on cuda_stream.
 *
 * Returns 0; -1 invalid argument (null pointer, non-positive dimension, negative batch, a restriction above, a
 * workspace limit below one item); -5 a CUDA call failed -- su2_ozaki_last_error() names it.  batch == 0 is a no-op. */
int32_t su2_gemm_pair_batched_i8(int32_t m, int32_t k, int32_t n, int32_t p, int64_t batch, double alpha,
                                 const double* A, const double* X, const double* B, double* C, int32_t nslices,
                                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* One product on its own, C_b (m x n) = A_b (m x k) * X_b (k x n) (overwritten, no alpha): the unit the oracle's
 * emulated_matmul defines, for element-by-element parity.  Same restriction. */
int32_t su2_matmul_batched_i8(int32_t m, int32_t k, int32_t n, int64_t batch, const double* A, const double* X,
                              double* C, int32_t nslices, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* out = H_eff * psi with every task of a plan executed on the INT8 tensor path (row f4 inside the hot path):
 * tasks: HOST [ntask], the records that su2_heff.h's export of task views hands out (device operands of the plan).
 * Per task F_s += coef * sum_pos alpha_pos * Aop_pos * E * Dop_pos^T (Eq. (3)) runs as two batched sliced
 * products over the positions: E is sliced once per task, A_pos / D_pos on the fly (operators stored transposed become
 * MN-major INT8 operands, no transposed copy; a block shared by all positions is sliced once), the second product's
 * integer planes are recombined and summed over the positions in index order (deterministic) into F_s.
 * psi, out: DEVICE [psi_len] (out is overwritten; must not alias psi).  workspace: DEVICE, 256-byte aligned; a task is
 * processed in chunks of as many positions as fit (about 7 (m k + p n + m n) + 28 m max(n, p) bytes per position).
 * Accuracy: each product within the bound above with K = k or n; 7 slices give <= 1e-12 of max|F| on the synthetic
 * workloads (tests: 1e-10 against the oracle, the tolerance of su2_heff_apply).  Launch-bound for small blocks: one task
 * costs 17 + 2 kernel launches, so this pays for bonds whose blocks hold several hundred multiplets.
 * Returns 0, -1 (invalid argument, a contraction too long for exact int32 sums, workspace below one position) or -5. */
int32_t su2_heff_apply_i8(const su2_task_view* tasks, int64_t ntask, const double* psi, double* out, int64_t psi_len,
                          int32_t nslices, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Bytes of workspace `items` items need (p = 0: the single product); 0 for invalid arguments. */
size_t su2_ozaki_workspace_bytes(int32_t m, int32_t k, int32_t n, int32_t p, int64_t items, int32_t nslices);

/* Kernels this library has launched since load (bench.py's gpu_launches). */
int64_t su2_ozaki_launch_count(void);

/* Text of the calling thread's last error ("" if none). */
const char* su2_ozaki_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
