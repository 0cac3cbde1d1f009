// Persistent fp64 DP5 guiding-centre tracer: one particle per thread, warp-aggregated refill
// from a global work counter (PAPER.md:57-61 for what is computed; the launch shape is this
// library's own, not the paper's 64-thread/8-particle blocks of PAPER.md:59).
#include "gc_device.cuh"

namespace catapult {

constexpr int TRACE_THREADS = 128;

template <int MODEL>
__global__ void __launch_bounds__(TRACE_THREADS)
trace_kernel(const __grid_constant__ TraceConst tc, const __grid_constant__ TraceArgs a) {
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const long long n = a.n;

  // per-lane particle state (registers)
  double y[4], k1[4], t = 0.0, dt = 0.0, mu = 0.0;
  long long idx = -1;
  unsigned nacc = 0, nrej = 0;
  long long attempts_left = 0;
  int consecutive = 0;
  bool active = false, exhausted = false;
  // per-lane statistics
  unsigned long long c_acc = 0, c_rej = 0, c_eval = 0;
  unsigned c_fin[4] = {0, 0, 0, 0};

  for (;;) {
    // ---- refill: lanes without a particle pull the next index (one atomic per warp) ----------
    const unsigned need = __ballot_sync(FULL, !active && !exhausted);
    if (need) {
      const int leader = __ffs(need) - 1;
      unsigned long long base = 0;
      if (lane == leader) base = atomicAdd(a.queue, (unsigned long long)__popc(need));
      base = __shfl_sync(FULL, base, leader);
      if (!active && !exhausted) {
        const long long mine = (long long)base + __popc(need & ((1u << lane) - 1u));
        if (mine >= n) {
          exhausted = true;
        } else {
          idx = mine;
          double x[4];
#pragma unroll
          for (int c = 0; c < 4; ++c) x[c] = a.x_in[c * n + idx];
          bool skip = false;
          if (a.resume) {
            skip = (a.status[idx] != CATAPULT_ST_REACHED_T);
            t = a.t_io[idx];
            if (!(t < tc.T)) skip = true;  // already at (or past) the requested end time
          } else {
            t = 0.0;
          }
          if (!skip) {
            state_to_y<MODEL>(x, y);
            double B, level;
            // mu needs |B| at the start point; the same evaluation then gives k1
            double dy0[4];
            rhs<MODEL>(tc, t, y, 0.0, dy0, B, level);
            ++c_eval;
            if (a.resume) {
              mu = a.mu_io[idx];
              dt = a.dt_io[idx];
            } else {
              mu = (tc.vtot2 - x[3] * x[3]) / (2.0 * B);
              dt = tc.dt0;
            }
            if (!a.resume && is_lost<MODEL>(tc, level)) {
              // born outside: returned unchanged, t_stop = 0
#pragma unroll
              for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = x[c];
              a.t_io[idx] = 0.0;
              a.status[idx] = CATAPULT_ST_LOST;
              if (a.dt_io) a.dt_io[idx] = dt;
              if (a.mu_io) a.mu_io[idx] = mu;
              if (a.nacc) a.nacc[idx] = 0;
              if (a.nrej) a.nrej[idx] = 0;
              ++c_fin[CATAPULT_ST_LOST];
            } else if (a.init_only) {
              a.t_io[idx] = 0.0;
              a.status[idx] = CATAPULT_ST_REACHED_T;
              a.dt_io[idx] = dt;
              a.mu_io[idx] = mu;
            } else {
              rhs<MODEL>(tc, t, y, mu, k1, B, level);
              ++c_eval;
              nacc = 0;
              nrej = 0;
              consecutive = 0;
              attempts_left = tc.max_steps > 0 ? tc.max_steps : -1;
              active = true;
            }
          }
        }
      }
    }
    if (!__any_sync(FULL, active)) {
      if (__all_sync(FULL, exhausted)) break;
      continue;
    }

    // ---- one attempted step for every active lane ----------------------------------------------
    if (active) {
      int finish = -1;
      if (attempts_left == 0) {
        finish = CATAPULT_ST_MAXSTEPS;
      } else {
        const double rem = tc.T - t;
        const bool clamped = !(dt < rem);  // the last step lands exactly on T (S4)
        const double h = clamped ? rem : dt;
        double ynew[4], k7[4], err[4], level;
        dp5_attempt<MODEL, false>(tc, t, y, k1, h, mu, ynew, k7, err, level, nullptr);
        c_eval += 6;
        if (attempts_left > 0) --attempts_left;
        const double r = error_ratio(tc, err, y, k1, h);
        bool accepted;
        const double dtn = controller(h, r, tc.dtmax, accepted);
        if (!accepted) {
          ++nrej;
          dt = dtn;
          if (++consecutive >= tc.max_rej) finish = CATAPULT_ST_STALLED;  // DESIGN.md S6
        } else {
          consecutive = 0;
          ++nacc;
          t = clamped ? tc.T : t + h;
          if (!clamped) dt = dtn;
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            y[i] = ynew[i];
            k1[i] = k7[i];
          }
          // DESIGN.md S5: loss first, then T
          if (is_lost<MODEL>(tc, level)) finish = CATAPULT_ST_LOST;
          else if (t >= tc.T) finish = CATAPULT_ST_REACHED_T;
        }
      }
      if (finish >= 0) {
        double x[4];
        y_to_state<MODEL>(y, x);
#pragma unroll
        for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = x[c];
        a.t_io[idx] = t;
        a.status[idx] = finish;
        if (a.dt_io) a.dt_io[idx] = dt;
        if (a.mu_io) a.mu_io[idx] = mu;
        if (a.nacc) a.nacc[idx] = (a.resume ? a.nacc[idx] : 0u) + nacc;
        if (a.nrej) a.nrej[idx] = (a.resume ? a.nrej[idx] : 0u) + nrej;
        c_acc += nacc;
        c_rej += nrej;
        ++c_fin[finish];
        active = false;
      }
    }
  }

  // ---- statistics: warp-reduce, one atomic per warp per counter ----------------------------------
  if (a.counters) {
    unsigned long long v[7] = {c_acc, c_rej, c_fin[0], c_fin[1], c_fin[2], c_fin[3], c_eval};
#pragma unroll
    for (int j = 0; j < 7; ++j) {
      unsigned long long s = v[j];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
      if (lane == 0 && s) atomicAdd(a.counters + j, s);
    }
  }
}

template <int MODEL>
__global__ void step_once_kernel(const __grid_constant__ TraceConst tc, long long n, const double* __restrict__ d_x,
                                 const double* __restrict__ d_t, const double* __restrict__ d_h,
                                 double* __restrict__ d_xnew, double* __restrict__ d_err, double* __restrict__ d_k) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double x[4], y[4], k1[4], ynew[4], k7[4], err[4], kall[28], B, level;
#pragma unroll
  for (int c = 0; c < 4; ++c) x[c] = d_x[c * n + i];
  state_to_y<MODEL>(x, y);
  const double t = d_t[i], h = d_h[i];
  rhs<MODEL>(tc, t, y, 0.0, k1, B, level);
  const double mu = (tc.vtot2 - x[3] * x[3]) / (2.0 * B);
  rhs<MODEL>(tc, t, y, mu, k1, B, level);
  dp5_attempt<MODEL, true>(tc, t, y, k1, h, mu, ynew, k7, err, level, kall);
  double xn[4];
  y_to_state<MODEL>(ynew, xn);
#pragma unroll
  for (int c = 0; c < 4; ++c) d_xnew[c * n + i] = xn[c];
  d_err[i] = error_ratio(tc, err, y, k1, h);
#pragma unroll
  for (int j = 0; j < 28; ++j) d_k[(long long)j * n + i] = kall[j];
}

template <int MODEL>
static catapult_status shape_for(int64_t n, int* blocks, int* threads) {
  int dev = 0, sms = 0, per_sm = 0;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  CATAPULT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  CATAPULT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_kernel<MODEL>, TRACE_THREADS, 0));
  if (per_sm < 1) per_sm = 1;
  long long resident = (long long)sms * per_sm;
  long long want = (n + TRACE_THREADS - 1) / TRACE_THREADS;
  if (want < 1) want = 1;
  *blocks = (int)(want < resident ? want : resident);
  *threads = TRACE_THREADS;
  return CATAPULT_OK;
}

catapult_status trace_launch_shape(int model, int64_t n, int* blocks, int* threads) {
  switch (model) {
    case MODEL_BOOZER_VAC: return shape_for<MODEL_BOOZER_VAC>(n, blocks, threads);
    case MODEL_BOOZER_SAW: return shape_for<MODEL_BOOZER_SAW>(n, blocks, threads);
    default: return shape_for<MODEL_CART>(n, blocks, threads);
  }
}

catapult_status launch_trace(const TraceConst& tc, const TraceArgs& a, int model, cudaStream_t s) {
  if (a.n == 0) return CATAPULT_OK;
  int blocks = 0, threads = 0;
  catapult_status st = trace_launch_shape(model, a.n, &blocks, &threads);
  if (st != CATAPULT_OK) return st;
  switch (model) {
    case MODEL_BOOZER_VAC: trace_kernel<MODEL_BOOZER_VAC><<<blocks, threads, 0, s>>>(tc, a); break;
    case MODEL_BOOZER_SAW: trace_kernel<MODEL_BOOZER_SAW><<<blocks, threads, 0, s>>>(tc, a); break;
    default: trace_kernel<MODEL_CART><<<blocks, threads, 0, s>>>(tc, a); break;
  }
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

catapult_status launch_step_once(const TraceConst& tc, int model, int64_t n, const double* d_x, const double* d_t,
                                 const double* d_h, double* d_xnew, double* d_err, double* d_k, cudaStream_t s) {
  if (n == 0) return CATAPULT_OK;
  const int threads = 64;
  const int blocks = (int)((n + threads - 1) / threads);
  switch (model) {
    case MODEL_BOOZER_VAC:
      step_once_kernel<MODEL_BOOZER_VAC><<<blocks, threads, 0, s>>>(tc, n, d_x, d_t, d_h, d_xnew, d_err, d_k);
      break;
    case MODEL_BOOZER_SAW:
      step_once_kernel<MODEL_BOOZER_SAW><<<blocks, threads, 0, s>>>(tc, n, d_x, d_t, d_h, d_xnew, d_err, d_k);
      break;
    default:
      step_once_kernel<MODEL_CART><<<blocks, threads, 0, s>>>(tc, n, d_x, d_t, d_h, d_xnew, d_err, d_k);
      break;
  }
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

}  // namespace catapult
