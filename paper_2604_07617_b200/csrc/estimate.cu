// Monte-Carlo estimate phi_hat = (1/n) sum g(Y_i) (Eq. 2) as a deterministic two-pass
// device reduction: fixed block partition, fixed-order tree inside a block, fixed-order final sum.
#include "internal.h"

namespace catapult {

constexpr int EST_THREADS = 256;
constexpr int EST_MAX_BLOCKS = 1024;

__device__ __forceinline__ double g_of(int g_kind, long long i, const int* status, const double* tstop,
                                       const double* g_user) {
  if (g_kind == 0) return status[i] == CATAPULT_ST_LOST ? 1.0 : 0.0;
  if (g_kind == 1) return tstop[i];
  return g_user[i];
}

__global__ void __launch_bounds__(EST_THREADS)
estimate_partial_kernel(int g_kind, long long n, const int* __restrict__ status, const double* __restrict__ tstop,
                        const double* __restrict__ g_user, double* __restrict__ partial /*[gridDim.x][2]*/) {
  __shared__ double s1[EST_THREADS], s2[EST_THREADS];
  // contiguous chunk per block, strided inside the block: the partition depends only on (n, grid)
  const long long per_block = (n + gridDim.x - 1) / gridDim.x;
  const long long lo = (long long)blockIdx.x * per_block;
  const long long hi = lo + per_block < n ? lo + per_block : n;
  double a = 0.0, b = 0.0;
  for (long long i = lo + threadIdx.x; i < hi; i += EST_THREADS) {
    const double g = g_of(g_kind, i, status, tstop, g_user);
    a += g;
    b = fma(g, g, b);
  }
  s1[threadIdx.x] = a;
  s2[threadIdx.x] = b;
  __syncthreads();
  for (int o = EST_THREADS / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      s1[threadIdx.x] += s1[threadIdx.x + o];
      s2[threadIdx.x] += s2[threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    partial[2 * blockIdx.x] = s1[0];
    partial[2 * blockIdx.x + 1] = s2[0];
  }
}

__global__ void estimate_final_kernel(long long n, int nblocks, const double* __restrict__ partial,
                                      double* __restrict__ out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double sum = 0.0, sum2 = 0.0;
  for (int b = 0; b < nblocks; ++b) {
    sum += partial[2 * b];
    sum2 += partial[2 * b + 1];
  }
  const double mean = n > 0 ? sum / (double)n : 0.0;
  double var = n > 1 ? (sum2 / (double)n - mean * mean) / (double)(n - 1) : 0.0;
  if (var < 0.0) var = 0.0;
  out[0] = mean;
  out[1] = sqrt(var);
  out[2] = sum;
  out[3] = sum2;
}

catapult_status launch_estimate(int g_kind, int64_t n, const int* d_status, const double* d_tstop, const double* d_g,
                                double* d_out, cudaStream_t s) {
  long long want = (n + EST_THREADS * 8 - 1) / (EST_THREADS * 8);
  int blocks = (int)(want < 1 ? 1 : (want > EST_MAX_BLOCKS ? EST_MAX_BLOCKS : want));
  double* partial = nullptr;
  CATAPULT_CUDA_TRY(cudaMallocAsync((void**)&partial, sizeof(double) * 2 * blocks, s));
  estimate_partial_kernel<<<blocks, EST_THREADS, 0, s>>>(g_kind, n, d_status, d_tstop, d_g, partial);
  estimate_final_kernel<<<1, 32, 0, s>>>(n, blocks, partial, d_out);
  cudaError_t e = cudaGetLastError();
  cudaFreeAsync(partial, s);
  CATAPULT_CUDA_TRY(e);
  return CATAPULT_OK;
}

// ---- catapult_estimate_static: the same estimate for callers that are not allowed to allocate ---------------------
// (include/catapult.h has the user-facing contract).  The per-block partial sums, which launch_estimate() above keeps
// in a stream-ordered allocation, live here in an array that is part of the loaded library image: 16 KiB on every
// GPU that loads libcatapult.so, held until the process exits, shared by every call on that GPU.
//
// Two things about this array are easy to get wrong:
//  * In HOST code the name `estimate_static_scratch` is only a handle for the runtime, not a device address; handing
//    it to a kernel makes the kernel fault (or scribble over host memory on systems where the GPU can reach it).
//    The device address has to be asked for with cudaGetSymbolAddress, with the device in question current, and it is
//    different on every device.  estimate_static_scratch_ptr() below does that once per device and remembers it.
//  * Nothing here must start at zero: estimate_partial_kernel writes every slot [0, 2*blocks) that
//    estimate_final_kernel reads, so whatever an earlier call left behind is never seen.
constexpr int EST_STATIC_MAX_DEVICES = 64;
static __device__ __align__(256) double estimate_static_scratch[2 * EST_MAX_BLOCKS];

static_assert(CATAPULT_ESTIMATE_STATIC_MAX_N == (long long)EST_MAX_BLOCKS * EST_THREADS * 8,
              "catapult.h's limit = one scratch slot per block of EST_THREADS * 8 particles");

// Device address of the scratch array on the CURRENT device; looked up on the first call per device (no allocation:
// cudaGetSymbolAddress only reports where the already loaded image put the array), cached afterwards.
static catapult_status estimate_static_scratch_ptr(double** out) {
  static double* cache[EST_STATIC_MAX_DEVICES] = {};  // written once per device; a racing duplicate writes the same value
  int dev = -1;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  if (dev >= 0 && dev < EST_STATIC_MAX_DEVICES) {
    double* c = __atomic_load_n(&cache[dev], __ATOMIC_ACQUIRE);
    if (c) {
      *out = c;
      return CATAPULT_OK;
    }
  }
  double* p = nullptr;
  CATAPULT_CUDA_TRY(cudaGetSymbolAddress((void**)&p, estimate_static_scratch));
  if (!p) {
    set_error("cudaGetSymbolAddress(estimate_static_scratch) returned a null address");
    return CATAPULT_ECUDA;
  }
  if (dev >= 0 && dev < EST_STATIC_MAX_DEVICES) __atomic_store_n(&cache[dev], p, __ATOMIC_RELEASE);
  *out = p;
  return CATAPULT_OK;
}

catapult_status launch_estimate_static(int g_kind, int64_t n, const int* d_status, const double* d_tstop,
                                       const double* d_g, double* d_out, cudaStream_t s) {
  if (n > CATAPULT_ESTIMATE_STATIC_MAX_N) {
    set_error("catapult_estimate_static: n exceeds CATAPULT_ESTIMATE_STATIC_MAX_N (2097152 particles, the size its "
              "built-in scratch array was made for); use catapult_estimate, which allocates its scratch");
    return CATAPULT_EINVAL;
  }
  // the block partition of launch_estimate() for the same n (never capped below the limit above), so both entry
  // points add the same numbers in the same order
  const long long want = (n + EST_THREADS * 8 - 1) / (EST_THREADS * 8);
  const int blocks = (int)(want < 1 ? 1 : want);
  double* partial = nullptr;
  catapult_status st = estimate_static_scratch_ptr(&partial);
  if (st != CATAPULT_OK) return st;
  estimate_partial_kernel<<<blocks, EST_THREADS, 0, s>>>(g_kind, n, d_status, d_tstop, d_g, partial);
  estimate_final_kernel<<<1, 32, 0, s>>>(n, blocks, partial, d_out);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

}  // namespace catapult
