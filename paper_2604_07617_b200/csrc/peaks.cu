// Roofline denominators measured on the device in use: the sustained
// DFMA rate of all SMs and the L2 read bandwidth.  MEASURED_PEAKS.json carries neither.
#include "internal.h"

namespace catapult {

// 16 independent DFMA chains per thread, 256 threads per block, several blocks per SM.
__global__ void __launch_bounds__(256) dfma_kernel(double* out, int iters, double seed) {
  double a[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) a[j] = seed + j * 1e-3 + threadIdx.x * 1e-6;
  const double m = 1.0000001, c = 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < 16; ++j) a[j] = fma(a[j], m, c);
  }
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < 16; ++j) s += a[j];
  if (s == 123.456) out[0] = s;  // keeps the chains alive
}

catapult_status measure_fp64_peak(double* flops) {
  int dev = 0, sms = 0;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  CATAPULT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double* d = nullptr;
  CATAPULT_CUDA_TRY(cudaMalloc((void**)&d, sizeof(double)));
  cudaEvent_t e0, e1;
  CATAPULT_CUDA_TRY(cudaEventCreate(&e0));
  CATAPULT_CUDA_TRY(cudaEventCreate(&e1));
  const int blocks = sms * 8, threads = 256, iters = 20000;
  dfma_kernel<<<blocks, threads>>>(d, 2000, 1.0);  // warm-up
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    dfma_kernel<<<blocks, threads>>>(d, iters, 1.0);
    cudaEventRecord(e1);
    CATAPULT_CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * 16.0 * (double)iters * threads * blocks / (ms * 1e-3);
    if (fl > best) best = fl;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  *flops = best;
  return CATAPULT_OK;
}

__global__ void __launch_bounds__(512) l2_read_kernel(const double2* __restrict__ buf, long long nvec, int passes,
                                                      double* out) {
  double acc = 0.0;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (int p = 0; p < passes; ++p) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
      double2 v;
      asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(buf + i));
      acc += v.x + v.y;
    }
  }
  if (acc == 123.456) out[0] = acc;
}

catapult_status measure_l2_bandwidth(size_t bytes, double* bps) {
  int dev = 0, sms = 0;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  CATAPULT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (bytes < 4096) bytes = 4096;
  bytes &= ~(size_t)15;
  double* d = nullptr;
  CATAPULT_CUDA_TRY(cudaMalloc((void**)&d, bytes + sizeof(double)));
  CATAPULT_CUDA_TRY(cudaMemset(d, 0, bytes + sizeof(double)));
  const long long nvec = (long long)(bytes / 16);
  cudaEvent_t e0, e1;
  CATAPULT_CUDA_TRY(cudaEventCreate(&e0));
  CATAPULT_CUDA_TRY(cudaEventCreate(&e1));
  const int blocks = sms * 4, threads = 512, passes = 64;
  double* sink = d + bytes / 8;
  l2_read_kernel<<<blocks, threads>>>((const double2*)d, nvec, 2, sink);  // warm the L2
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    l2_read_kernel<<<blocks, threads>>>((const double2*)d, nvec, passes, sink);
    cudaEventRecord(e1);
    CATAPULT_CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double b = (double)bytes * passes / (ms * 1e-3);
    if (b > best) best = b;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  *bps = best;
  return CATAPULT_OK;
}

}  // namespace catapult
