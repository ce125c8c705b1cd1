// Measurement aid, built as its OWN library (libsu2probe.so, include/su2_probe.h) so that nothing of it ships in the
// product ABI: register-resident FP64 throughput of this GPU, with which bench.py quotes the roofline denominator it
// measured itself (MEASURED_PEAKS.json has no FP64 entry).  kind 0: DFMA loop; kind 1: mma.sync m8n8k4 f64 (SASS
// DMMA.8x8x4) loop.
#include <cuda_runtime.h>

#include "su2_probe.h"

namespace {
__global__ void __launch_bounds__(256) dfma_probe(double* out, int iters, double a, double b) {
  double x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(256) dmma_probe(double* out, int iters, double a, double b) {
  double c[8][2];
#pragma unroll
  for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
  if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace

extern "C" int32_t su2_probe_fp64_peak(int32_t kind, int32_t iters, int32_t ctas_per_sm, double* tflops, void* cuda_stream) {
  if (!tflops || iters <= 0 || ctas_per_sm <= 0 || (kind != 0 && kind != 1)) return -1;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return -5;
  double* buf = nullptr;
  const int grid = sms * ctas_per_sm;
  if (cudaMalloc(&buf, (size_t)grid * 256 * sizeof(double)) != cudaSuccess) return -5;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    if (kind == 0) dfma_probe<<<grid, 256, 0, st>>>(buf, iters, 1.0000001, 1e-9);
    else dmma_probe<<<grid, 256, 0, st>>>(buf, iters, 1.0000001, 1e-9);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(buf); return -5; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(buf);
  const double flops = kind == 0 ? (double)grid * 256 * (double)iters * 16 * 2
                                 : (double)grid * 8 /*warps*/ * (double)iters * 8 * (2.0 * 8 * 8 * 4);
  *tflops = flops / (best * 1e-3) / 1e12;
  return 0;
}
