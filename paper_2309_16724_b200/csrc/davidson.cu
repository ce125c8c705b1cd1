// Davidson eigensolver around su2_heff_apply ("iterative
// diagonalization ... via the Lanczos or Davidson algorithms").  The paper gives no algorithmic
// detail; reading G8:
//   * Rayleigh-Ritz in a subspace of at most max_subspace vectors, restart from the Ritz vector when full;
//   * new direction t = r / (diag - theta) ONLY while theta lies below min(diag) by a margin (the Newton-like
//     diagonal correction is then positive definite); otherwise the plain Krylov direction t = r.  With theta
//     inside the range of diag the quotient collapses to spikes on the few elements whose diag is close to
//     theta and the iteration stalls (measured in round 1: |r| flat over 20 steps at configs[2]);
//   * classical Gram-Schmidt applied twice (one batched projection + one update per pass).
// Everything between the apply and the two scalars handed back runs on the device, stream-ordered: the k x k
// Rayleigh-Ritz problem (k <= 64) is diagonalised by ONE CTA with a parallel-ordered cyclic Jacobi, coefficients
// stay in device memory, and a step synchronises once, at its end, for (theta, |r|).  BLAS-1 parts use fixed-grid
// two-stage reductions (deterministic).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <vector>

#include "su2_internal.h"


#define SU2_CUDA(call)                                   \
  do {                                                   \
    cudaError_t _e = (call);                             \
    if (_e != cudaSuccess) {                             \
      su2::set_cuda_error(#call, (int)_e);               \
      return SU2_ERR_CUDA;                               \
    }                                                    \
  } while (0)

namespace {

constexpr int RED_BLOCKS = 296;    // 2 per SM; fixed so that sums are reproducible
constexpr int RED_THREADS = 256;
constexpr int MAX_SUB = 64;
// layout of the small device state behind the reduction scratch (doubles)
constexpr int ST_G = 0;                          // MAX_SUB x MAX_SUB projected matrix G = V^T H V (leading dimension MAX_SUB)
constexpr int ST_Y = ST_G + MAX_SUB * MAX_SUB;   // Ritz vector in the subspace
constexpr int ST_C = ST_Y + MAX_SUB;             // Gram-Schmidt projections / norms
constexpr int ST_RES = ST_C + MAX_SUB;           // [theta, |r|^2, min(diag), max(diag)]
constexpr int ST_SIZE = ST_RES + 8;

// partial[j][b] = sum over block b's stripe of x_j[i]*y[i]  (j = blockIdx.y)
__global__ void __launch_bounds__(RED_THREADS)
dot_stage1(const double* __restrict__ xs, int64_t xstride, const double* __restrict__ y, int64_t n, double* __restrict__ partial) {
  __shared__ double sm[RED_THREADS];
  const double* x = xs + (int64_t)blockIdx.y * xstride;
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)RED_BLOCKS * RED_THREADS) s += x[i] * y[i];
  sm[threadIdx.x] = s;
  __syncthreads();
  for (int w = RED_THREADS / 2; w > 0; w >>= 1) {
    if (threadIdx.x < w) sm[threadIdx.x] += sm[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[(int64_t)blockIdx.y * RED_BLOCKS + blockIdx.x] = sm[0];
}
// result j = sum_b partial[j][b], stored at out1[j * s1] and (if out2) out2[j * s2]
__global__ void __launch_bounds__(RED_THREADS)
dot_stage2(const double* __restrict__ partial, double* __restrict__ out1, int s1, double* __restrict__ out2, int s2) {
  __shared__ double sm[RED_THREADS];
  double s = 0.0;
  for (int i = threadIdx.x; i < RED_BLOCKS; i += RED_THREADS) s += partial[(int64_t)blockIdx.x * RED_BLOCKS + i];
  sm[threadIdx.x] = s;
  __syncthreads();
  for (int w = RED_THREADS / 2; w > 0; w >>= 1) {
    if (threadIdx.x < w) sm[threadIdx.x] += sm[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    out1[(int64_t)blockIdx.x * s1] = sm[0];
    if (out2) out2[(int64_t)blockIdx.x * s2] = sm[0];
  }
}
// min and max of x (two-stage, one launch each)
__global__ void __launch_bounds__(RED_THREADS)
minmax_stage1(const double* __restrict__ x, int64_t n, double* __restrict__ partial) {
  __shared__ double lo[RED_THREADS], hi[RED_THREADS];
  double a = INFINITY, b = -INFINITY;
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)RED_BLOCKS * RED_THREADS) {
    a = fmin(a, x[i]);
    b = fmax(b, x[i]);
  }
  lo[threadIdx.x] = a; hi[threadIdx.x] = b;
  __syncthreads();
  for (int w = RED_THREADS / 2; w > 0; w >>= 1) {
    if (threadIdx.x < w) {
      lo[threadIdx.x] = fmin(lo[threadIdx.x], lo[threadIdx.x + w]);
      hi[threadIdx.x] = fmax(hi[threadIdx.x], hi[threadIdx.x + w]);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { partial[2 * blockIdx.x] = lo[0]; partial[2 * blockIdx.x + 1] = hi[0]; }
}
__global__ void __launch_bounds__(RED_THREADS)
minmax_stage2(const double* __restrict__ partial, double* __restrict__ out) {
  __shared__ double lo[RED_THREADS], hi[RED_THREADS];
  double a = INFINITY, b = -INFINITY;
  for (int i = threadIdx.x; i < RED_BLOCKS; i += RED_THREADS) { a = fmin(a, partial[2 * i]); b = fmax(b, partial[2 * i + 1]); }
  lo[threadIdx.x] = a; hi[threadIdx.x] = b;
  __syncthreads();
  for (int w = RED_THREADS / 2; w > 0; w >>= 1) {
    if (threadIdx.x < w) {
      lo[threadIdx.x] = fmin(lo[threadIdx.x], lo[threadIdx.x + w]);
      hi[threadIdx.x] = fmax(hi[threadIdx.x], hi[threadIdx.x + w]);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = lo[0]; out[1] = hi[0]; }
}

// Rayleigh-Ritz on the device: lowest eigenpair of the k x k symmetric matrix G (leading dimension MAX_SUB).
// One CTA.  Cyclic Jacobi in the round-robin ("tournament") order: a sweep is K-1 rounds of K/2 rotations on
// disjoint index pairs, which commute and are applied together -- columns (and the eigenvector matrix) by all
// threads, then rows.  Sweeps stop when the off-diagonal mass is below 1e-30 of the Frobenius norm.
// Output: y[0..k) = eigenvector of the lowest eigenvalue (sign: largest component positive), res[0] = theta.
__global__ void __launch_bounds__(256)
ritz_kernel(const double* __restrict__ G, int k, double* __restrict__ y, double* __restrict__ res) {
  extern __shared__ double ritz_smem[];              // a, v: K x (K + 1) each
  const int K = (k + 1) & ~1;                       // even number of players; index k (if k is odd) sits out
  const int LD = K + 1;
  double* a_ = ritz_smem;
  double* v_ = ritz_smem + K * LD;
#define a(i, j) a_[(i) * LD + (j)]
#define v(i, j) v_[(i) * LD + (j)]
  __shared__ double cs[MAX_SUB / 2][2];
  __shared__ int pq[MAX_SUB / 2][2];
  __shared__ double red[256];
  __shared__ int s_lo;
  const int tid = threadIdx.x;
  for (int e = tid; e < K * K; e += 256) {
    const int i = e / K, j = e % K;
    a(i, j) = (i < k && j < k) ? G[i * MAX_SUB + j] : 0.0;
    v(i, j) = (i == j) ? 1.0 : 0.0;
  }
  __syncthreads();
  for (int sweep = 0; sweep < 30; ++sweep) {
    double off = 0.0, tot = 0.0;
    for (int e = tid; e < k * k; e += 256) {
      const int i = e / k, j = e % k;
      const double x = a(i, j) * a(i, j);
      tot += x;
      if (i != j) off += x;
    }
    red[tid] = off;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) { if (tid < w) red[tid] += red[tid + w]; __syncthreads(); }
    off = red[0];
    __syncthreads();
    red[tid] = tot;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) { if (tid < w) red[tid] += red[tid + w]; __syncthreads(); }
    tot = red[0];
    __syncthreads();
    if (off <= 1e-30 * tot || k < 2) break;
    for (int round = 0; round < K - 1; ++round) {
      if (tid < K / 2) {
        // circle method: player K-1 is fixed, the others rotate
        int p, q;
        if (tid == 0) { p = K - 1; q = (K - 1 - round) % (K - 1); }
        else { p = (tid + (K - 1) - round % (K - 1)) % (K - 1); q = ((K - 1 - tid) + (K - 1) - round % (K - 1)) % (K - 1); }
        if (p > q) { const int t = p; p = q; q = t; }
        double c = 1.0, s = 0.0;
        if (q < k) {
          const double apq = a(p, q);
          if (fabs(apq) > 1e-300) {
            const double tau = (a(q, q) - a(p, p)) / (2.0 * apq);
            const double t = (tau >= 0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
            c = 1.0 / sqrt(1.0 + t * t);
            s = t * c;
          }
        }
        pq[tid][0] = p; pq[tid][1] = q; cs[tid][0] = c; cs[tid][1] = s;
      }
      __syncthreads();
      for (int e = tid; e < K * (K / 2); e += 256) {       // A <- A J, V <- V J
        const int i = e / (K / 2), r = e % (K / 2);
        const int p = pq[r][0], q = pq[r][1];
        const double c = cs[r][0], s = cs[r][1];
        const double aip = a(i, p), aiq = a(i, q);
        a(i, p) = c * aip - s * aiq;
        a(i, q) = s * aip + c * aiq;
        const double vip = v(i, p), viq = v(i, q);
        v(i, p) = c * vip - s * viq;
        v(i, q) = s * vip + c * viq;
      }
      __syncthreads();
      for (int e = tid; e < K * (K / 2); e += 256) {       // A <- J^T A
        const int i = e / (K / 2), r = e % (K / 2);
        const int p = pq[r][0], q = pq[r][1];
        const double c = cs[r][0], s = cs[r][1];
        const double api = a(p, i), aqi = a(q, i);
        a(p, i) = c * api - s * aqi;
        a(q, i) = s * api + c * aqi;
      }
      __syncthreads();
    }
  }
  if (tid == 0) {
    int lo = 0;
    for (int i = 1; i < k; ++i)
      if (a(i, i) < a(lo, lo)) lo = i;
    s_lo = lo;
    res[0] = a(lo, lo);
  }
  __syncthreads();
  const int lo = s_lo;
  if (tid == 0) {
    int big = 0;
    for (int i = 1; i < k; ++i)
      if (fabs(v(i, lo)) > fabs(v(big, lo))) big = i;
    red[0] = v(big, lo) < 0.0 ? -1.0 : 1.0;
  }
  __syncthreads();
  if (tid < MAX_SUB) y[tid] = tid < k ? red[0] * v(tid, lo) : 0.0;
#undef a
#undef v
}

// out = sum_j c[j] * (a_j - shift * b_j), c = y (device), shift = res[0] (device) if b, else out = sum_j c[j] a_j.
// With `partial`: also the block-partial sums of out^2 (stage 1 of |out|^2; grid must be RED_BLOCKS x RED_THREADS).
__global__ void __launch_bounds__(RED_THREADS)
lincomb_dev(double* __restrict__ out, const double* __restrict__ a, const double* __restrict__ b, int64_t stride, int k,
            const double* __restrict__ y, const double* __restrict__ res, int64_t n, double* __restrict__ partial) {
  __shared__ double c[MAX_SUB];
  __shared__ double sm[RED_THREADS];
  if (threadIdx.x < k) c[threadIdx.x] = y[threadIdx.x];
  __syncthreads();
  const double shift = b ? res[0] : 0.0;
  double ss = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double s = 0.0;
    for (int j = 0; j < k; ++j) {
      double v = a[(int64_t)j * stride + i];
      if (b) v -= shift * b[(int64_t)j * stride + i];
      s += c[j] * v;
    }
    out[i] = s;
    ss += s * s;
  }
  if (partial) {
    sm[threadIdx.x] = ss;
    __syncthreads();
    for (int w = RED_THREADS / 2; w > 0; w >>= 1) {
      if (threadIdx.x < w) sm[threadIdx.x] += sm[threadIdx.x + w];
      __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sm[0];
  }
}
// Gram-Schmidt update t -= sum_j c[j] V_j with the projections c left on the device by dot_stage2
__global__ void __launch_bounds__(256)
gs_update(double* __restrict__ t, const double* __restrict__ V, int64_t stride, int k, const double* __restrict__ cdev, int64_t n) {
  __shared__ double c[MAX_SUB];
  if (threadIdx.x < k) c[threadIdx.x] = cdev[threadIdx.x];
  __syncthreads();
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double s = t[i];
    for (int j = 0; j < k; ++j) s -= c[j] * V[(int64_t)j * stride + i];
    t[i] = s;
  }
}
// y = x / sqrt(c[0]) (0 if c[0] == 0)
__global__ void __launch_bounds__(256) scale_copy_rnorm_dev(double* __restrict__ y, const double* __restrict__ x, const double* __restrict__ c, int64_t n) {
  const double nrm = sqrt(c[0]);
  const double a = nrm > 0 ? 1.0 / nrm : 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) y[i] = a * x[i];
}
__global__ void __launch_bounds__(256) copy2(double* __restrict__ y0, const double* __restrict__ x0, double* __restrict__ y1,
                                             const double* __restrict__ x1, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    y0[i] = x0[i];
    if (y1) y1[i] = x1[i];
  }
}
// New direction (reading G8): res = [theta, |r|^2, min(diag), max(diag)].  While theta < min(diag) - margin the
// diagonal correction t = r / (diag - theta) (all denominators positive, >= margin); otherwise t = r.
__global__ void __launch_bounds__(256)
precondition(double* __restrict__ t, const double* __restrict__ r, const double* __restrict__ diag, const double* __restrict__ res,
             int mode, int64_t n) {
  const double theta = res[0], dmin = res[2], dmax = res[3];
  const double margin = 1e-3 * fmax(dmax - dmin, 1e-300) + 1e-12 * fmax(fabs(dmin), fabs(dmax));
  const bool use_diag = mode == 1 && theta < dmin - margin;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    t[i] = use_diag ? r[i] / (diag[i] - theta) : r[i];
}
// after a restart the subspace is {Ritz vector}: G = [theta], y = [1]
__global__ void restart_state(double* __restrict__ st) {
  const int i = threadIdx.x + blockIdx.x * blockDim.x;
  if (i < MAX_SUB * MAX_SUB) st[ST_G + i] = (i == 0) ? st[ST_RES] : 0.0;
  if (i < MAX_SUB) st[ST_Y + i] = (i == 0) ? 1.0 : 0.0;
}

}  // namespace

struct su2_davidson {
  int64_t n = 0;
  int32_t mmax = 0, k = 0;      // k basis vectors V[0..k), W computed for [0..k-1)
  int32_t ky = 0;               // valid entries of the Ritz vector y (device)
  double *V = nullptr, *W = nullptr, *diag = nullptr, *r = nullptr, *t = nullptr, *u = nullptr, *scratch = nullptr;
  double* state = nullptr;      // device: G, y, Gram-Schmidt coefficients, [theta, |r|^2, min diag, max diag]
  double* h_result = nullptr;   // pinned
  int32_t precond_mode = 1;     // 1: diagonal correction when theta < min(diag) (else Krylov); 0: always Krylov
  int32_t grid = 296;
  su2_reduce_fn reduce = nullptr;   // position-sharded plans: sums a vector over the ranks (null: single GPU)
  void* reduce_user = nullptr;
};

// orthogonalise d->t against V[0..k) (classical Gram-Schmidt, twice), normalise into V[k]; stream-ordered
static su2_status orthonormalise_into_basis(su2_davidson* d, cudaStream_t st) {
  double* cdev = d->state + ST_C;
  const int k = d->k;
  for (int pass = 0; pass < 2 && k > 0; ++pass) {
    dim3 g1(RED_BLOCKS, k);
    dot_stage1<<<g1, RED_THREADS, 0, st>>>(d->V, d->n, d->t, d->n, d->scratch);
    dot_stage2<<<k, RED_THREADS, 0, st>>>(d->scratch, cdev, 1, nullptr, 0);
    gs_update<<<d->grid, 256, 0, st>>>(d->t, d->V, d->n, k, cdev, d->n);
    su2::count_launch(3);
  }
  dot_stage1<<<dim3(RED_BLOCKS, 1), RED_THREADS, 0, st>>>(d->t, d->n, d->t, d->n, d->scratch);
  dot_stage2<<<1, RED_THREADS, 0, st>>>(d->scratch, cdev, 1, nullptr, 0);
  scale_copy_rnorm_dev<<<d->grid, 256, 0, st>>>(d->V + (int64_t)k * d->n, d->t, cdev, d->n);
  su2::count_launch(3);
  SU2_CUDA(cudaGetLastError());
  d->k += 1;
  return SU2_OK;
}

extern "C" int64_t su2_davidson_workspace_bytes(const su2_plan* plan, int32_t max_subspace) {
  if (!plan || max_subspace < 2 || max_subspace > MAX_SUB) return -1;
  const int64_t n = plan->psi_len;
  return (2 * (int64_t)max_subspace + 4) * n * 8 + ((int64_t)MAX_SUB * RED_BLOCKS + ST_SIZE) * 8 + 256;
}

extern "C" su2_status su2_davidson_create(su2_davidson** out, const su2_plan* plan, int32_t max_subspace, const double* x0_dev,
                                          void* ws, void* cuda_stream) {
  return su2_davidson_create_sharded(out, plan, max_subspace, x0_dev, ws, cuda_stream, nullptr, nullptr);
}

extern "C" su2_status su2_davidson_create_sharded(su2_davidson** out, const su2_plan* plan, int32_t max_subspace,
                                                  const double* x0_dev, void* ws, void* cuda_stream, su2_reduce_fn reduce,
                                                  void* reduce_user) {
  if (!out || !plan || !x0_dev || !ws || max_subspace < 2 || max_subspace > MAX_SUB) return SU2_ERR_INVALID_ARGUMENT;
  if (plan->host_only) return SU2_ERR_NO_DEVICE_PLAN;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  su2_davidson* d = new su2_davidson();
  d->n = plan->psi_len;
  d->mmax = max_subspace;
  d->reduce = reduce;
  d->reduce_user = reduce_user;
  const int64_t n = plan->psi_len;
  double* base = (double*)ws;
  d->V = base;
  d->W = d->V + (int64_t)max_subspace * n;
  d->diag = d->W + (int64_t)max_subspace * n;
  d->r = d->diag + n;
  d->t = d->r + n;
  d->u = d->t + n;
  d->scratch = d->u + n;
  d->state = d->scratch + (int64_t)MAX_SUB * RED_BLOCKS;
  d->grid = 2 * plan->num_sms;
  if (cudaMallocHost(&d->h_result, 8 * sizeof(double)) != cudaSuccess) {
    delete d;
    return SU2_ERR_CUDA;
  }
  if (cudaFuncSetAttribute(ritz_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)(2 * MAX_SUB * (MAX_SUB + 1) * sizeof(double))) != cudaSuccess) { su2_davidson_destroy(d); return SU2_ERR_CUDA; }
  if (cudaMemsetAsync(d->state, 0, ST_SIZE * sizeof(double), st) != cudaSuccess) { su2_davidson_destroy(d); return SU2_ERR_CUDA; }
  su2_status s = su2_heff_diag(plan, d->diag, cuda_stream);
  if (s == SU2_OK && d->reduce) s = d->reduce(d->diag, d->n, cuda_stream, d->reduce_user);   // diag of a sum of shards
  if (s != SU2_OK) { su2_davidson_destroy(d); return s; }
  minmax_stage1<<<RED_BLOCKS, RED_THREADS, 0, st>>>(d->diag, d->n, d->scratch);
  minmax_stage2<<<1, RED_THREADS, 0, st>>>(d->scratch, d->state + ST_RES + 2);
  // first basis vector = x0 / |x0|
  copy2<<<d->grid, 256, 0, st>>>(d->t, x0_dev, nullptr, nullptr, d->n);
  su2::count_launch(3);
  d->k = 0;
  s = orthonormalise_into_basis(d, st);
  if (s != SU2_OK) { su2_davidson_destroy(d); return s; }
  *out = d;
  return SU2_OK;
}

extern "C" su2_status su2_davidson_set_preconditioner(su2_davidson* d, int32_t mode) {
  if (!d || mode < 0 || mode > 1) return SU2_ERR_INVALID_ARGUMENT;
  d->precond_mode = mode;
  return SU2_OK;
}

extern "C" su2_status su2_davidson_step(const su2_plan* plan, su2_davidson* d, void* workspace_dev, void* cuda_stream,
                                        double* theta_out, double* resnorm_out) {
  if (!plan || !d || !theta_out || !resnorm_out || d->k < 1) return SU2_ERR_INVALID_ARGUMENT;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int k = d->k, mm = d->mmax;
  const int64_t n = d->n;
  double* G = d->state + ST_G;
  double* y = d->state + ST_Y;
  double* res = d->state + ST_RES;
  // 1. w = H_eff v for the newest basis vector
  su2_status s = su2_heff_apply(plan, d->V + (int64_t)(k - 1) * n, d->W + (int64_t)(k - 1) * n, workspace_dev, cuda_stream);
  if (s != SU2_OK) return s;
  // 1b. position-sharded plan: this rank applied its share of the positions; sum F over the ranks (the path's one
  //     exchange step).  Every rank receives the same bits, so the replicated algebra below stays in step.
  if (d->reduce) {
    s = d->reduce(d->W + (int64_t)(k - 1) * n, n, cuda_stream, d->reduce_user);
    if (s != SU2_OK) return s;
  }
  // 2. new row and column of the projected matrix G = V^T H V (device)
  dot_stage1<<<dim3(RED_BLOCKS, k), RED_THREADS, 0, st>>>(d->V, n, d->W + (int64_t)(k - 1) * n, n, d->scratch);
  dot_stage2<<<k, RED_THREADS, 0, st>>>(d->scratch, G + (k - 1), MAX_SUB, G + (int64_t)(k - 1) * MAX_SUB, 1);
  // 3. Rayleigh-Ritz in the k-dimensional subspace (one CTA): y, theta
  {
    const int K = (k + 1) & ~1;
    ritz_kernel<<<1, 256, 2 * K * (K + 1) * sizeof(double), st>>>(G, k, y, res);
  }
  d->ky = k;
  // 4. residual r = sum_i y_i (W_i - theta V_i) and |r|^2
  lincomb_dev<<<RED_BLOCKS, RED_THREADS, 0, st>>>(d->r, d->W, d->V, n, k, y, res, n, d->scratch);
  dot_stage2<<<1, RED_THREADS, 0, st>>>(d->scratch, res + 1, 1, nullptr, 0);
  // 5. new direction
  precondition<<<d->grid, 256, 0, st>>>(d->t, d->r, d->diag, res, d->precond_mode, n);
  su2::count_launch(6);
  SU2_CUDA(cudaMemcpyAsync(d->h_result, res, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
  // 6. restart from the Ritz vector when the subspace is full: V <- {V y}, W <- {W y}, G <- {theta}
  if (k == mm) {
    lincomb_dev<<<RED_BLOCKS, RED_THREADS, 0, st>>>(d->r, d->V, nullptr, n, k, y, res, n, nullptr);
    lincomb_dev<<<RED_BLOCKS, RED_THREADS, 0, st>>>(d->u, d->W, nullptr, n, k, y, res, n, nullptr);
    copy2<<<d->grid, 256, 0, st>>>(d->V, d->r, d->W, d->u, n);
    restart_state<<<(MAX_SUB * MAX_SUB + 255) / 256, 256, 0, st>>>(d->state);
    su2::count_launch(4);
    SU2_CUDA(cudaGetLastError());
    d->k = 1;
    d->ky = 1;
  }
  // 7. orthonormalise and append
  s = orthonormalise_into_basis(d, st);
  if (s != SU2_OK) return s;
  SU2_CUDA(cudaGetLastError());
  // the step's only synchronisation: the two scalars handed back
  SU2_CUDA(cudaStreamSynchronize(st));
  *theta_out = d->h_result[0];
  *resnorm_out = std::sqrt(std::fmax(d->h_result[1], 0.0));
  return SU2_OK;
}

extern "C" su2_status su2_davidson_ritz_vector(const su2_davidson* d, double* x_dev, void* cuda_stream) {
  if (!d || !x_dev || d->ky < 1) return SU2_ERR_INVALID_ARGUMENT;
  lincomb_dev<<<RED_BLOCKS, RED_THREADS, 0, (cudaStream_t)cuda_stream>>>(x_dev, d->V, nullptr, d->n, d->ky, d->state + ST_Y,
                                                                         d->state + ST_RES, d->n, nullptr);
  su2::count_launch();
  SU2_CUDA(cudaGetLastError());
  return SU2_OK;
}

extern "C" su2_status su2_davidson_destroy(su2_davidson* d) {
  if (!d) return SU2_ERR_INVALID_ARGUMENT;
  if (d->h_result) cudaFreeHost(d->h_result);
  delete d;
  return SU2_OK;
}
