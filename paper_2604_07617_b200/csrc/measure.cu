// Measurements g on the END states of a trace other than the loss indicator and the stop time (PAPER.md:25:
// "Similar functions g can be chosen to calculate energy loss ..., wall-loads from alpha particles"; DESIGN.md
// readings G2, G3).  Both kernels read the trace's outputs once: HBM-bound, one thread per particle, coalesced
// structure-of-arrays reads; the lost-energy kernel adds one table evaluation (a 512-byte block per quantity) for
// every LOST particle.
#include "gc_device.cuh"
#include "gc_math.cuh"

namespace catapult {

constexpr int MEASURE_THREADS = 256;

// Reading G2: g_i = 1[lost] (vpar^2 / 2 + mu |B|(x_f)) / (v_total^2 / 2).  |B| from the table in the one evaluation
// order every user of the table follows (horner64): Boozer column 0; cylindrical sqrt(B_R^2 + B_phi^2 + B_Z^2).
template <bool BOOZER>
__global__ void __launch_bounds__(MEASURE_THREADS)
lost_energy_kernel(const __grid_constant__ FieldConst f, double inv_E0, long long n, const double* __restrict__ xf,
                   const double* __restrict__ mu, const int* __restrict__ status, double* __restrict__ g) {
  using AX = AxisRoles<BOOZER>;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (status[i] != CATAPULT_ST_LOST) {
    g[i] = 0.0;
    return;
  }
  const double x0 = xf[i], x1 = xf[n + i], x2 = xf[2 * n + i], vpar = xf[3 * n + i];
  double w[3], B;
  if (BOOZER) {
    const int cell = locate<true>(f, x0, x1, x2, w);
    const double* src = f.table + (long long)cell * f.m * 64;  // column 0 = |B| (also in derivative-of-interpolant mode)
    B = horner64([&](int e, double& f0, double& f1, double& f2, double& f3) { ldg_f64x4(src + e, f0, f1, f2, f3); },
                 w[AX::LAST], w[AX::SECOND], w[AX::FIRST]);
  } else {
    const double R = ::sqrt(fma(x0, x0, x1 * x1));
    const int cell = locate<false>(f, R, x2, fm::atan2(x1, x0), w);
    double b2 = 0.0;
#pragma unroll 1
    for (int q = 0; q < 3; ++q) {  // B_R, B_phi, B_Z
      const double* src = f.table + ((long long)cell * f.m + q) * 64;
      const double v = horner64(
          [&](int e, double& f0, double& f1, double& f2, double& f3) { ldg_f64x4(src + e, f0, f1, f2, f3); },
          w[AX::LAST], w[AX::SECOND], w[AX::FIRST]);
      b2 = fma(v, v, b2);
    }
    B = ::sqrt(b2);
  }
  g[i] = fma(mu[i], B, 0.5 * vpar * vpar) * inv_E0;
}

// one histogram bin, the operations of the oracle's orc_bin one by one (no contraction: the bin is an integer that
// floating point decides): u = (a - lo) / span, reduced to [0, 1) when periodic, floor(u nb) clamped to [0, nb - 1]
__device__ __forceinline__ int exit_bin(double a, double lo, double span, bool periodic, int nb) {
  double u = __ddiv_rn(__dsub_rn(a, lo), span);
  if (periodic) u = __dsub_rn(u, floor(u));
  const double b = floor(__dmul_rn(u, (double)nb));
  return b < 0.0 ? 0 : (b > (double)(nb - 1) ? nb - 1 : (int)b);   // NaN -> bin 0
}

// Reading G3: lost particles per bin of the exit point.  Integer counts: atomic adds commute, the result does not
// depend on the order.  Boozer: (theta, zeta), both periodic; cylindrical: (phi = atan2(y, x) periodic, Z clamped).
template <bool BOOZER>
__global__ void __launch_bounds__(MEASURE_THREADS)
exit_histogram_kernel(const __grid_constant__ FieldConst f, long long n, const double* __restrict__ xf,
                      const int* __restrict__ status, int nb0, int nb1, unsigned long long* __restrict__ hist) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n || status[i] != CATAPULT_ST_LOST) return;
  int b0, b1;
  if (BOOZER) {
    b0 = exit_bin(xf[n + i], f.lo[1], f.span[1], true, nb0);
    b1 = exit_bin(xf[2 * n + i], f.lo[2], f.span[2], true, nb1);
  } else {
    b0 = exit_bin(::atan2(xf[n + i], xf[i]), f.lo[2], f.span[2], true, nb0);
    b1 = exit_bin(xf[2 * n + i], f.lo[1], f.span[1], false, nb1);
  }
  atomicAdd(hist + (long long)b0 * nb1 + b1, 1ull);
}

catapult_status launch_lost_energy(const FieldConst& fc, double inv_E0, int64_t n, const double* d_xf, const double* d_mu,
                                   const int* d_status, double* d_g, cudaStream_t s) {
  if (n == 0) return CATAPULT_OK;
  const int blocks = (int)((n + MEASURE_THREADS - 1) / MEASURE_THREADS);
  if (fc.coord == CATAPULT_COORD_BOOZER)
    lost_energy_kernel<true><<<blocks, MEASURE_THREADS, 0, s>>>(fc, inv_E0, n, d_xf, d_mu, d_status, d_g);
  else
    lost_energy_kernel<false><<<blocks, MEASURE_THREADS, 0, s>>>(fc, inv_E0, n, d_xf, d_mu, d_status, d_g);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

catapult_status launch_exit_histogram(const FieldConst& fc, int64_t n, const double* d_xf, const int* d_status, int nb0,
                                      int nb1, unsigned long long* d_hist, cudaStream_t s) {
  CATAPULT_CUDA_TRY(cudaMemsetAsync(d_hist, 0, sizeof(unsigned long long) * (size_t)nb0 * nb1, s));
  if (n == 0) return CATAPULT_OK;
  const int blocks = (int)((n + MEASURE_THREADS - 1) / MEASURE_THREADS);
  if (fc.coord == CATAPULT_COORD_BOOZER)
    exit_histogram_kernel<true><<<blocks, MEASURE_THREADS, 0, s>>>(fc, n, d_xf, d_status, nb0, nb1, d_hist);
  else
    exit_histogram_kernel<false><<<blocks, MEASURE_THREADS, 0, s>>>(fc, n, d_xf, d_status, nb0, nb1, d_hist);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

}  // namespace catapult
