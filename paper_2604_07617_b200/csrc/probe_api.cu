// C-ABI entry points of libcatapult_probe.so (include/catapult_probe.h): measurement and test hooks kept out of
// the product library.
#include <cstdio>

#include "catapult_probe.h"
#include "internal.h"

namespace catapult {

static thread_local std::string g_probe_error;

void set_error(const std::string& msg) { g_probe_error = msg; }

catapult_status cuda_fail(cudaError_t e, const char* what) {
  char buf[512];
  std::snprintf(buf, sizeof(buf), "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
  set_error(buf);
  return e == cudaErrorMemoryAllocation ? CATAPULT_ENOMEM : CATAPULT_ECUDA;
}

static catapult_status fail(catapult_status st, const char* msg) {
  set_error(msg);
  return st;
}

}  // namespace catapult

using namespace catapult;

extern "C" {

const char* catapult_probe_last_error(void) { return g_probe_error.c_str(); }

catapult_status catapult_math_probe(int32_t fn, int64_t n, const double* d_a, const double* d_b, double* d_out0,
                                    double* d_out1, void* stream) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (fn < 0 || fn > CATAPULT_FN_CONTROLLER) return fail(CATAPULT_EINVAL, "unknown fn");
  if (n > 0 && (!d_a || !d_out0)) return fail(CATAPULT_EINVAL, "d_a/d_out0 is NULL");
  if (n > 0 && (fn == CATAPULT_FN_ATAN2 || fn == CATAPULT_FN_CONTROLLER) && !d_b)
    return fail(CATAPULT_EINVAL, "atan2 / controller need d_b");
  return launch_math_probe(fn, n, d_a, d_b, d_out0, d_out1, (cudaStream_t)stream);
}

catapult_status catapult_measure_fp64_peak(double* flops_per_s) {
  if (!flops_per_s) return fail(CATAPULT_EINVAL, "flops_per_s is NULL");
  return measure_fp64_peak(flops_per_s);
}

catapult_status catapult_measure_l2_bandwidth(size_t bytes, double* bytes_per_s) {
  if (!bytes_per_s) return fail(CATAPULT_EINVAL, "bytes_per_s is NULL");
  return measure_l2_bandwidth(bytes, bytes_per_s);
}

}  // extern "C"
