// Davidson eigensolver around su2_heff_apply ("iterative
// diagonalization ... via the Lanczos or Davidson algorithms").  The paper gives no algorithmic
// detail; reading G8: diagonal preconditioner t = r / (theta - diag) with |theta - diag|
// floored at 1e-8 * max|diag|, modified Gram-Schmidt applied twice, restart from the Ritz vector
// when the subspace is full.  BLAS-1 parts use fixed-grid two-stage reductions (deterministic).
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

struct Coefs { double c[MAX_SUB]; };

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
__global__ void __launch_bounds__(RED_THREADS)
dot_stage2(const double* __restrict__ partial, double* __restrict__ result) {
  __shared__ double sm[RED_THREADS];
  double s = 0.0;
  for (int i = threadIdx.x; i < RED_BLOCKS; i += RED_THREADS) s += partial[(int64_t)blockIdx.x * RED_BLOCKS + i];
  sm[threadIdx.x] = s;
  __syncthreads();
  for (int w = RED_THREADS / 2; w > 0; w >>= 1) {
    if (threadIdx.x < w) sm[threadIdx.x] += sm[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) result[blockIdx.x] = sm[0];
}
__global__ void __launch_bounds__(RED_THREADS)
maxabs_stage1(const double* __restrict__ x, int64_t n, double* __restrict__ partial) {
  __shared__ double sm[RED_THREADS];
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)RED_BLOCKS * RED_THREADS) s = fmax(s, fabs(x[i]));
  sm[threadIdx.x] = s;
  __syncthreads();
  for (int w = RED_THREADS / 2; w > 0; w >>= 1) {
    if (threadIdx.x < w) sm[threadIdx.x] = fmax(sm[threadIdx.x], sm[threadIdx.x + w]);
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = sm[0];
}
// out = sum_j c[j] * (a_j - shift * b_j)   (b may be null: out = sum_j c[j] a_j)
__global__ void __launch_bounds__(256)
lincomb(double* __restrict__ out, const double* __restrict__ a, const double* __restrict__ b, int64_t stride, int k, Coefs c,
        double shift, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double s = 0.0;
    for (int j = 0; j < k; ++j) {
      double v = a[(int64_t)j * stride + i];
      if (b) v -= shift * b[(int64_t)j * stride + i];
      s += c.c[j] * v;
    }
    out[i] = s;
  }
}
__global__ void __launch_bounds__(256) axpy(double* __restrict__ y, const double* __restrict__ x, double a, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) y[i] += a * x[i];
}
// the same two with the scalar left on the device by dot_stage2 (no host round trip inside Gram-Schmidt):
// y -= c[0] x, and y = x / sqrt(c[0]) (0 if c[0] == 0); same operations, same bits as the host-scalar versions
__global__ void __launch_bounds__(256) axpy_neg_dev(double* __restrict__ y, const double* __restrict__ x, const double* __restrict__ c, int64_t n) {
  const double a = -c[0];
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) y[i] += a * x[i];
}
__global__ void __launch_bounds__(256) scale_copy_rnorm_dev(double* __restrict__ y, const double* __restrict__ x, const double* __restrict__ c, int64_t n) {
  const double nrm = sqrt(c[0]);
  const double a = nrm > 0 ? 1.0 / nrm : 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) y[i] = a * x[i];
}
__global__ void __launch_bounds__(256) scale_copy(double* __restrict__ y, const double* __restrict__ x, double a, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) y[i] = a * x[i];
}
// t = r / (theta - diag), |theta - diag| floored at `floor_` keeping the sign
__global__ void __launch_bounds__(256)
precondition(double* __restrict__ t, const double* __restrict__ r, const double* __restrict__ diag, double theta, double floor_, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double den = theta - diag[i];
    if (fabs(den) < floor_) den = den < 0.0 ? -floor_ : floor_;
    t[i] = r[i] / den;
  }
}

// cyclic Jacobi eigen-decomposition of a small symmetric matrix (k <= 64): a -> eigenvalues, v columns
void jacobi_eigh(int k, std::vector<double>& a, std::vector<double>& v, std::vector<double>& w) {
  v.assign((size_t)k * k, 0.0);
  for (int i = 0; i < k; ++i) v[(size_t)i * k + i] = 1.0;
  for (int sweep = 0; sweep < 100; ++sweep) {
    double off = 0.0;
    for (int i = 0; i < k; ++i)
      for (int j = i + 1; j < k; ++j) off += a[(size_t)i * k + j] * a[(size_t)i * k + j];
    if (off < 1e-300) break;
    for (int p = 0; p < k; ++p)
      for (int q = p + 1; q < k; ++q) {
        const double apq = a[(size_t)p * k + q];
        if (std::fabs(apq) < 1e-300) continue;
        const double tau = (a[(size_t)q * k + q] - a[(size_t)p * k + p]) / (2.0 * apq);
        const double t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
        const double c = 1.0 / std::sqrt(1.0 + t * t), s = t * c;
        for (int i = 0; i < k; ++i) {
          const double aip = a[(size_t)i * k + p], aiq = a[(size_t)i * k + q];
          a[(size_t)i * k + p] = c * aip - s * aiq;
          a[(size_t)i * k + q] = s * aip + c * aiq;
        }
        for (int i = 0; i < k; ++i) {
          const double api = a[(size_t)p * k + i], aqi = a[(size_t)q * k + i];
          a[(size_t)p * k + i] = c * api - s * aqi;
          a[(size_t)q * k + i] = s * api + c * aqi;
        }
        for (int i = 0; i < k; ++i) {
          const double vip = v[(size_t)i * k + p], viq = v[(size_t)i * k + q];
          v[(size_t)i * k + p] = c * vip - s * viq;
          v[(size_t)i * k + q] = s * vip + c * viq;
        }
      }
  }
  w.resize(k);
  for (int i = 0; i < k; ++i) w[i] = a[(size_t)i * k + i];
}

}  // namespace

struct su2_davidson {
  int64_t n = 0;
  int32_t mmax = 0, k = 0;      // k basis vectors V[0..k), W computed for [0..k-1)
  double *V = nullptr, *W = nullptr, *diag = nullptr, *r = nullptr, *t = nullptr, *u = nullptr, *scratch = nullptr;
  double* h_result = nullptr;   // pinned
  std::vector<double> G;        // mmax x mmax projected matrix
  std::vector<double> y;        // last Ritz vector in the subspace
  double diag_floor = 0.0;
  int32_t grid = 296;
  su2_reduce_fn reduce = nullptr;   // position-sharded plans: sums a vector over the ranks (null: single GPU)
  void* reduce_user = nullptr;
};

static su2_status dots(su2_davidson* d, const double* xs, int nx, const double* y, double* host_out, cudaStream_t st) {
  dim3 g1(RED_BLOCKS, nx);
  dot_stage1<<<g1, RED_THREADS, 0, st>>>(xs, d->n, y, d->n, d->scratch); su2::count_launch();
  dot_stage2<<<nx, RED_THREADS, 0, st>>>(d->scratch, d->scratch + (int64_t)MAX_SUB * RED_BLOCKS); su2::count_launch();
  SU2_CUDA(cudaGetLastError());
  SU2_CUDA(cudaMemcpyAsync(d->h_result, d->scratch + (int64_t)MAX_SUB * RED_BLOCKS, nx * sizeof(double), cudaMemcpyDeviceToHost, st));
  SU2_CUDA(cudaStreamSynchronize(st));
  for (int i = 0; i < nx; ++i) host_out[i] = d->h_result[i];
  return SU2_OK;
}

// orthogonalise d->t against V[0..k) (modified Gram-Schmidt, twice), normalise into V[k]
static su2_status orthonormalise_into_basis(su2_davidson* d, cudaStream_t st) {
  // every scalar (projection, norm) stays on the device: the loop is stream-ordered, no synchronisation
  double* res = d->scratch + (int64_t)MAX_SUB * RED_BLOCKS;
  auto dot_dev = [&](const double* x, const double* y) {
    dim3 g1(RED_BLOCKS, 1);
    dot_stage1<<<g1, RED_THREADS, 0, st>>>(x, d->n, y, d->n, d->scratch); su2::count_launch();
    dot_stage2<<<1, RED_THREADS, 0, st>>>(d->scratch, res); su2::count_launch();
  };
  for (int pass = 0; pass < 2; ++pass)
    for (int i = 0; i < d->k; ++i) {
      dot_dev(d->V + (int64_t)i * d->n, d->t);
      axpy_neg_dev<<<d->grid, 256, 0, st>>>(d->t, d->V + (int64_t)i * d->n, res, d->n); su2::count_launch();
    }
  dot_dev(d->t, d->t);
  scale_copy_rnorm_dev<<<d->grid, 256, 0, st>>>(d->V + (int64_t)d->k * d->n, d->t, res, d->n); su2::count_launch();
  SU2_CUDA(cudaGetLastError());
  d->k += 1;
  return SU2_OK;
}

extern "C" int64_t su2_davidson_workspace_bytes(const su2_plan* plan, int32_t max_subspace) {
  if (!plan || max_subspace < 2 || max_subspace > MAX_SUB) return -1;
  const int64_t n = plan->psi_len;
  return (2 * (int64_t)max_subspace + 4) * n * 8 + ((int64_t)MAX_SUB * RED_BLOCKS + MAX_SUB) * 8 + 256;
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
  d->G.assign((size_t)max_subspace * max_subspace, 0.0);
  d->grid = 2 * plan->num_sms;
  if (cudaMallocHost(&d->h_result, MAX_SUB * sizeof(double)) != cudaSuccess) {
    delete d;
    return SU2_ERR_CUDA;
  }
  su2_status s = su2_heff_diag(plan, d->diag, cuda_stream);
  if (s == SU2_OK && d->reduce) s = d->reduce(d->diag, d->n, cuda_stream, d->reduce_user);   // diag of a sum of shards
  if (s != SU2_OK) { su2_davidson_destroy(d); return s; }
  maxabs_stage1<<<RED_BLOCKS, RED_THREADS, 0, st>>>(d->diag, d->n, d->scratch); su2::count_launch();
  std::vector<double> part(RED_BLOCKS);
  if (cudaMemcpyAsync(part.data(), d->scratch, RED_BLOCKS * sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess) {
    su2_davidson_destroy(d);
    return SU2_ERR_CUDA;
  }
  double mx = 0.0;
  for (double v : part) mx = std::fmax(mx, v);
  d->diag_floor = 1e-8 * (mx > 0 ? mx : 1.0);
  // first basis vector = x0 / |x0|
  scale_copy<<<d->grid, 256, 0, st>>>(d->t, x0_dev, 1.0, d->n); su2::count_launch();
  d->k = 0;
  s = orthonormalise_into_basis(d, st);
  if (s != SU2_OK) { su2_davidson_destroy(d); return s; }
  *out = d;
  return SU2_OK;
}

extern "C" su2_status su2_davidson_step(const su2_plan* plan, su2_davidson* d, void* workspace_dev, void* cuda_stream,
                                        double* theta_out, double* resnorm_out) {
  if (!plan || !d || !theta_out || !resnorm_out || d->k < 1) return SU2_ERR_INVALID_ARGUMENT;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int k = d->k, mm = d->mmax;
  const int64_t n = d->n;
  // 1. w = H_eff v for the newest basis vector
  su2_status s = su2_heff_apply(plan, d->V + (int64_t)(k - 1) * n, d->W + (int64_t)(k - 1) * n, workspace_dev, cuda_stream);
  if (s != SU2_OK) return s;
  // 1b. position-sharded plan: this rank applied its share of the positions; sum F over the ranks (the path's one
  //     exchange step).  Every rank receives the same bits, so the replicated algebra below stays in step.
  if (d->reduce) {
    s = d->reduce(d->W + (int64_t)(k - 1) * n, n, cuda_stream, d->reduce_user);
    if (s != SU2_OK) return s;
  }
  // 2. new column of the projected matrix G = V^T H V
  std::vector<double> col(k);
  s = dots(d, d->V, k, d->W + (int64_t)(k - 1) * n, col.data(), st);
  if (s != SU2_OK) return s;
  for (int i = 0; i < k; ++i) d->G[(size_t)i * mm + (k - 1)] = d->G[(size_t)(k - 1) * mm + i] = col[i];
  // 3. Rayleigh-Ritz in the k-dimensional subspace (host, Jacobi)
  std::vector<double> a((size_t)k * k), v, w;
  for (int i = 0; i < k; ++i)
    for (int j = 0; j < k; ++j) a[(size_t)i * k + j] = d->G[(size_t)i * mm + j];
  jacobi_eigh(k, a, v, w);
  int lo = 0;
  for (int i = 1; i < k; ++i)
    if (w[i] < w[lo]) lo = i;
  const double theta = w[lo];
  Coefs c{};
  d->y.assign(k, 0.0);
  for (int i = 0; i < k; ++i) c.c[i] = d->y[i] = v[(size_t)i * k + lo];
  // 4. residual r = sum_i y_i (W_i - theta V_i)
  lincomb<<<d->grid, 256, 0, st>>>(d->r, d->W, d->V, n, k, c, theta, n); su2::count_launch();
  double rr = 0.0;
  s = dots(d, d->r, 1, d->r, &rr, st);
  if (s != SU2_OK) return s;
  *theta_out = theta;
  *resnorm_out = std::sqrt(rr);
  // 5. preconditioned direction
  precondition<<<d->grid, 256, 0, st>>>(d->t, d->r, d->diag, theta, d->diag_floor, n); su2::count_launch();
  // 6. restart from the Ritz vector when the subspace is full: V <- {V y}, W <- {W y}, G <- {theta}
  if (k == mm) {
    lincomb<<<d->grid, 256, 0, st>>>(d->r, d->V, nullptr, n, k, c, 0.0, n); su2::count_launch();
    lincomb<<<d->grid, 256, 0, st>>>(d->u, d->W, nullptr, n, k, c, 0.0, n); su2::count_launch();
    scale_copy<<<d->grid, 256, 0, st>>>(d->V, d->r, 1.0, n); su2::count_launch();
    scale_copy<<<d->grid, 256, 0, st>>>(d->W, d->u, 1.0, n); su2::count_launch();
    SU2_CUDA(cudaGetLastError());
    std::fill(d->G.begin(), d->G.end(), 0.0);
    d->G[0] = theta;
    d->k = 1;
    d->y.assign(1, 1.0);
  }
  // 7. orthonormalise and append
  s = orthonormalise_into_basis(d, st);
  if (s != SU2_OK) return s;
  SU2_CUDA(cudaGetLastError());
  return SU2_OK;
}

extern "C" su2_status su2_davidson_ritz_vector(const su2_davidson* d, double* x_dev, void* cuda_stream) {
  if (!d || !x_dev || d->y.empty()) return SU2_ERR_INVALID_ARGUMENT;
  Coefs c{};
  for (size_t i = 0; i < d->y.size(); ++i) c.c[i] = d->y[i];
  lincomb<<<d->grid, 256, 0, (cudaStream_t)cuda_stream>>>(x_dev, d->V, nullptr, d->n, (int)d->y.size(), c, 0.0, d->n); su2::count_launch();
  SU2_CUDA(cudaGetLastError());
  return SU2_OK;
}

extern "C" su2_status su2_davidson_destroy(su2_davidson* d) {
  if (!d) return SU2_ERR_INVALID_ARGUMENT;
  if (d->h_result) cudaFreeHost(d->h_result);
  delete d;
  return SU2_OK;
}
