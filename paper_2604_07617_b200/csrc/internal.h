// Internal declarations shared by the translation units of libcatapult.so (not installed).
#pragma once

#include <cuda_runtime.h>

#include <cstdint>
#include <string>

#include "catapult.h"

namespace catapult {

// Field geometry + profile parameters as the kernels see them.  Passed by value as a
// __grid_constant__ kernel parameter, i.e. it lives in the constant bank (PAPER.md:65:
// "Data that is used by all threads is moved to constant memory").
struct FieldConst {
  const double* table;  // [cell][quantity][64], cell-major (include/catapult.h)
  const double* node0;  // device scalar: first node of column 0 (written by field_build_kernel)
  const double* prof;   // non-vacuum Boozer: [3][3 k0 + 1] = G, I, iota on the unique s-nodes; nullptr: scalars
  int coord, m;
  int k[3];
  double lo[3], invh[3], span[3], invspan[3];
  double G, invG, psi0, invpsi0, iota0, iota1;
};

struct TraceConst {
  FieldConst f;
  double M, invM, q, Moq, vtot, vtot2;
  double T, rtol, atol, dt0, dtmax;  // dt0 / dtmax <= 0: DESIGN.md S3 defaults, resolved on the device
  long long max_steps;
  int max_rej;
  int loss_time_mode;  // include/catapult.h
  int saw_m, saw_n;
  double saw_Phi0, saw_s0, saw_invw2, saw_omega, saw_inv_omG;
};

struct TraceArgs {
  long long n;
  const double* x_in;  // [4][n]
  double* x_out;       // [4][n]
  double* t_io;        // [n]; in only when resume
  double* dt_io;       // [n] or nullptr
  double* mu_io;       // [n] or nullptr
  int* status;         // [n]; in only when resume
  unsigned* nacc;      // nullable
  unsigned* nrej;      // nullable
  unsigned long long* counters;  // nullable, CATAPULT_NCOUNTERS entries
  unsigned long long* queue;     // TRACE_SCRATCH_BYTES, zero at launch: the work counter, then one int per SM
                                 // (how many blocks of the launch have started there)
  int resume;     // 1: continue from (t,dt,mu,status) arrays
  int init_only;  // 1: only fill (t,dt,mu,status)
  // scripted replay (catapult_trace_scripted): step sizes are read instead of controlled
  const double* script_h;  // [script_len][n]; a particle stops at the first h <= 0
  double* script_r;        // [script_len][n] error ratio of every scripted step (nullable)
  int script_len;
  double* kall;            // step-once hook: [7][4][n] stage derivatives
};

constexpr size_t TRACE_SCRATCH_BYTES = 8 + 4 * 1024;

void set_error(const std::string& msg);
catapult_status cuda_fail(cudaError_t e, const char* what);

#define CATAPULT_CUDA_TRY(expr)                                        \
  do {                                                                 \
    cudaError_t _e = (expr);                                           \
    if (_e != cudaSuccess) return ::catapult::cuda_fail(_e, #expr);    \
  } while (0)

// field.cu
catapult_status launch_field_build(const catapult_field_desc& d, const double* d_nodes, double* d_table,
                                   double* d_node0, cudaStream_t s);
catapult_status launch_field_eval(const FieldConst& fc, int64_t npts, const double* d_pts, double* d_out,
                                  cudaStream_t s);
catapult_status launch_field_export_rows(const FieldConst& fc, int64_t ncells, double* d_out, cudaStream_t s);

// tracer.cu (mode: 0 adaptive, 1 scripted replay, 2 one attempted step)
catapult_status launch_trace(const TraceConst& tc, const TraceArgs& a, int model, int mode, cudaStream_t s);
catapult_status trace_launch_shape(int model, bool doi, int64_t n, int* blocks, int* threads);

// estimate.cu
catapult_status launch_estimate(int g_kind, int64_t n, const int* d_status, const double* d_tstop,
                                const double* d_g, double* d_out, cudaStream_t s);
// same sums, partial results in the library's own static device array: no allocation (catapult_estimate_static)
catapult_status launch_estimate_static(int g_kind, int64_t n, const int* d_status, const double* d_tstop,
                                       const double* d_g, double* d_out, cudaStream_t s);

// measure.cu
catapult_status launch_lost_energy(const FieldConst& fc, double inv_E0, int64_t n, const double* d_xf, const double* d_mu,
                                   const int* d_status, double* d_g, cudaStream_t s);
catapult_status launch_exit_histogram(const FieldConst& fc, int64_t n, const double* d_xf, const int* d_status, int nb0,
                                      int nb1, unsigned long long* d_hist, cudaStream_t s);

// mathprobe.cu
catapult_status launch_math_probe(int fn, int64_t n, const double* d_a, const double* d_b, double* d_o0, double* d_o1,
                                  cudaStream_t s);

// peaks.cu
catapult_status measure_fp64_peak(double* flops);
catapult_status measure_l2_bandwidth(size_t bytes, double* bps);

}  // namespace catapult

struct catapult_field {
  catapult_field_desc desc;
  catapult::FieldConst fc;
  double* d_table;   // table_bytes of coefficients, followed by the node0 scalar
  size_t table_bytes;
  int64_t ncells;
  int device;
  cudaEvent_t built;  // recorded on the build stream after field_build_kernel
};
