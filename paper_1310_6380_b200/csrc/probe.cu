// Diagnostic: the FP64 roofline denominators of this GPU, measured with register-only loops (no memory traffic):
// DMMA (mma.sync.m8n8k4.f64, the FP64 tensor pipe the zgemm uses) and DFMA (the plain FP64 pipe S1/S7 use).
// MEASURED_PEAKS.json holds no FP64 figure, so bench.py measures it in the same run.
#include "bs_internal.cuh"

namespace {
__global__ void __launch_bounds__(256) dmma_peak_kernel(double *out, int iters) {
  double c[16][2];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i][0] = c[i][1] = 0.0;
  const double a = threadIdx.x * 1e-3, b = threadIdx.x * 2e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[i][0]), "+d"(c[i][1])
                   : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(256) dfma_peak_kernel(double *out, int iters) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = i;
  const double a = 1.0 + threadIdx.x * 1e-9, b = threadIdx.x * 2e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace

extern "C" bs_status bs_fp64_peak(double *dmma_tflops, double *dfma_tflops, void *stream) {
  if (!dmma_tflops || !dfma_tflops) return BS_ERR_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return BS_ERR_CUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int blocks = sms * 2, threads = 256;
  double *out = nullptr;
  if (cudaMalloc(&out, sizeof(double) * blocks * threads) != cudaSuccess) return BS_ERR_CUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float ms = 0.f;
  const int iters = 40000;  // ~10 ms each
  dmma_peak_kernel<<<blocks, threads, 0, s>>>(out, 200);
  cudaEventRecord(e0, s);
  dmma_peak_kernel<<<blocks, threads, 0, s>>>(out, iters);
  cudaEventRecord(e1, s);
  cudaEventSynchronize(e1);
  cudaEventElapsedTime(&ms, e0, e1);
  *dmma_tflops = (double)blocks * (threads / 32) * iters * 16.0 * 512.0 / (ms * 1e9);
  dfma_peak_kernel<<<blocks, threads, 0, s>>>(out, 200);
  cudaEventRecord(e0, s);
  dfma_peak_kernel<<<blocks, threads, 0, s>>>(out, iters * 4);
  cudaEventRecord(e1, s);
  cudaEventSynchronize(e1);
  cudaEventElapsedTime(&ms, e0, e1);
  *dfma_tflops = (double)blocks * threads * iters * 4.0 * 16.0 * 2.0 / (ms * 1e9);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  return cudaGetLastError() == cudaSuccess ? BS_OK : BS_ERR_CUDA;
}
