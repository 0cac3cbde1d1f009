// Test hook: evaluates the device-side elementary functions of gc_math.cuh on arrays, so that
// tests/test_gpu_parity.py can compare them with numpy on the argument ranges the tracer uses.
#include "gc_device.cuh"
#include "catapult_probe.h"
#include "internal.h"

namespace catapult {

__global__ void math_probe_kernel(int fn, long long n, const double* __restrict__ a, const double* __restrict__ b,
                                  double* __restrict__ o0, double* __restrict__ o1) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const double x = a[i], y = b ? b[i] : 0.0;
    double r0 = 0.0, r1 = 0.0;
    switch (fn) {
      case CATAPULT_FN_ATAN2: r0 = fm::atan2(x, y); break;
      case CATAPULT_FN_SINCOS: fm::sincos(x, r0, r1); break;
      case CATAPULT_FN_EXP: r0 = fm::exp(x); break;
      case CATAPULT_FN_SQRT_RSQRT: fm::sqrt_rsqrt(x, r0, r1); break;
      case CATAPULT_FN_RCP: r0 = fm::rcp(x); break;
      case CATAPULT_FN_POW_NEG_INV: r0 = fm::pow_neg_inv(x, true); r1 = fm::pow_neg_inv(x, false); break;
      case CATAPULT_FN_CONTROLLER: {  // the tracer's step-size controller for an attempted step of length 1
        bool accepted;
        r0 = controller(1.0, x, y, accepted);
        r1 = accepted ? 1.0 : 0.0;
        break;
      }
      default: break;
    }
    o0[i] = r0;
    if (o1) o1[i] = r1;
  }
}

catapult_status launch_math_probe(int fn, int64_t n, const double* d_a, const double* d_b, double* d_o0, double* d_o1,
                                  cudaStream_t s) {
  if (n == 0) return CATAPULT_OK;
  long long blocks = (n + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  math_probe_kernel<<<(int)blocks, 256, 0, s>>>(fn, n, d_a, d_b, d_o0, d_o1);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

}  // namespace catapult
