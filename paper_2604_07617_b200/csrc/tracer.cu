// Persistent fp64 DP5 guiding-centre tracer (PAPER.md:57-61 for what is computed; the launch shape
// is this library's own, not the paper's 64-thread/8-particle blocks of PAPER.md:59).
//
// One particle per GROUP of NL lanes (gc_device.cuh), the current cell's coefficients cached in
// registers + shared memory, and a warp-aggregated refill from a global work counter so that groups
// whose particle is lost or finished pull the next one instead of idling.
#include "gc_device.cuh"

namespace catapult {

template <int MODEL, bool SCRIPT>
__global__ void __launch_bounds__(ModelTraits<MODEL>::NT, ModelTraits<MODEL>::MINB)
trace_kernel(const __grid_constant__ TraceConst tc, const __grid_constant__ TraceArgs a) {
  using MT = ModelTraits<MODEL>;
  constexpr int NL = MT::NL, CPL = MT::CPL;
  extern __shared__ double2 smem[];
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const long long n = a.n;
  const Group<NL> g;
  CellCache<MODEL> cc;
  cc.init(smem);

  // per-group particle state, replicated in the group's lanes (registers) except k1m
  double y[4], k1m[CPL], t = 0.0, dt = 0.0, mu = 0.0;
  long long idx = -1;
  unsigned nacc = 0, nrej = 0;
  long long attempts_left = 0;
  int consecutive = 0, step = 0;
  bool active = false, exhausted = false;
  // statistics (counted by every lane, reduced from lane 0 of each group)
  unsigned long long c_acc = 0, c_rej = 0, c_eval = 0;
  unsigned c_fin[4] = {0, 0, 0, 0};

  for (;;) {
    // ---- refill: groups without a particle pull the next index (one atomic per warp) ---------
    const bool want = !active && !exhausted;
    const unsigned need = __ballot_sync(FULL, want && g.j == 0);
    if (need) {
      const int leader = __ffs(need) - 1;
      unsigned long long base = 0;
      if (lane == leader) base = atomicAdd(a.queue, (unsigned long long)__popc(need));
      base = __shfl_sync(FULL, base, leader);
      if (want) {
        const long long mine = (long long)base + __popc(need & ((1u << g.gbase) - 1u));
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
            double B, level, dy0[4];
            // mu needs |B| at the start point; the same evaluation then gives k1
            rhs<MODEL>(tc, g, cc, t, y, 0.0, dy0, B, level);
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
              if (g.j == 0) {
#pragma unroll
                for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = x[c];
                a.t_io[idx] = 0.0;
                a.status[idx] = CATAPULT_ST_LOST;
                if (a.dt_io) a.dt_io[idx] = dt;
                if (a.mu_io) a.mu_io[idx] = mu;
                if (a.nacc) a.nacc[idx] = 0;
                if (a.nrej) a.nrej[idx] = 0;
              }
              ++c_fin[CATAPULT_ST_LOST];
            } else if (a.init_only) {
              if (g.j == 0) {
                a.t_io[idx] = 0.0;
                a.status[idx] = CATAPULT_ST_REACHED_T;
                a.dt_io[idx] = dt;
                a.mu_io[idx] = mu;
              }
            } else {
              rhs<MODEL>(tc, g, cc, t, y, mu, dy0, B, level);
              ++c_eval;
#pragma unroll
              for (int i = 0; i < CPL; ++i) k1m[i] = pick<NL>(dy0, i, g.j);
              nacc = 0;
              nrej = 0;
              consecutive = 0;
              step = 0;
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

    // ---- one attempted step for every active group ---------------------------------------------
    if (active) {
      int finish = -1;
      double h = 0.0;
      bool clamped = false;
      if (SCRIPT) {
        h = (step < a.script_len) ? a.script_h[(long long)step * n + idx] : 0.0;
        if (!(h > 0.0)) finish = CATAPULT_ST_REACHED_T;
      } else if (attempts_left == 0) {
        finish = CATAPULT_ST_MAXSTEPS;
      } else {
        const double rem = tc.T - t;
        clamped = !(dt < rem);  // the last step lands exactly on T (S4)
        h = clamped ? rem : dt;
      }
      if (finish < 0) {
        double ynew[4], k7m[CPL], errm[CPL], level;
        dp5_attempt<MODEL, false>(tc, g, cc, t, y, k1m, h, mu, ynew, k7m, errm, level, nullptr);
        c_eval += 6;
        if (attempts_left > 0) --attempts_left;
        const double r = error_ratio<NL, CPL>(tc, g, errm, y, k1m, h);
        bool accepted;
        double dtn;
        if (SCRIPT) {
          if (a.script_r && g.j == 0) a.script_r[(long long)step * n + idx] = r;
          ++step;
          accepted = true;
          dtn = h;
        } else {
          dtn = controller(h, r, tc.dtmax, accepted);
        }
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
          for (int i = 0; i < 4; ++i) y[i] = ynew[i];
#pragma unroll
          for (int i = 0; i < CPL; ++i) k1m[i] = k7m[i];
          // DESIGN.md S5: loss first, then T
          if (is_lost<MODEL>(tc, level)) finish = CATAPULT_ST_LOST;
          else if (!SCRIPT && t >= tc.T) finish = CATAPULT_ST_REACHED_T;
        }
      }
      if (finish >= 0) {
        if (g.j == 0) {
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
        }
        c_acc += nacc;
        c_rej += nrej;
        ++c_fin[finish];
        active = false;
      }
    }
  }

  // ---- statistics: warp-reduce over the group leaders, one atomic per warp per counter ---------------
  if (a.counters) {
    unsigned long long v[7] = {c_acc, c_rej, c_fin[0], c_fin[1], c_fin[2], c_fin[3], c_eval};
#pragma unroll
    for (int j = 0; j < 7; ++j) {
      unsigned long long s = (g.j == 0) ? v[j] : 0ull;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
      if (lane == 0 && s) atomicAdd(a.counters + j, s);
    }
  }
}

// test hook: one attempted step per particle, all seven stage derivatives
template <int MODEL>
__global__ void __launch_bounds__(ModelTraits<MODEL>::NT, ModelTraits<MODEL>::MINB)
step_once_kernel(const __grid_constant__ TraceConst tc, long long n, const double* __restrict__ d_x,
                 const double* __restrict__ d_t, const double* __restrict__ d_h, double* __restrict__ d_xnew,
                 double* __restrict__ d_err, double* __restrict__ d_k) {
  using MT = ModelTraits<MODEL>;
  constexpr int NL = MT::NL, CPL = MT::CPL;
  extern __shared__ double2 smem[];
  const Group<NL> g;
  CellCache<MODEL> cc;
  cc.init(smem);
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / NL;
  if (i >= n) return;  // group-uniform
  double x[4], y[4], dy[4], k1m[CPL], ynew[4], k7m[CPL], errm[CPL], kall_m[7 * CPL], B, level;
#pragma unroll
  for (int c = 0; c < 4; ++c) x[c] = d_x[c * n + i];
  state_to_y<MODEL>(x, y);
  const double t = d_t[i], h = d_h[i];
  rhs<MODEL>(tc, g, cc, t, y, 0.0, dy, B, level);
  const double mu = (tc.vtot2 - x[3] * x[3]) / (2.0 * B);
  rhs<MODEL>(tc, g, cc, t, y, mu, dy, B, level);
#pragma unroll
  for (int c = 0; c < CPL; ++c) k1m[c] = pick<NL>(dy, c, g.j);
  dp5_attempt<MODEL, true>(tc, g, cc, t, y, k1m, h, mu, ynew, k7m, errm, level, kall_m);
  const double r = error_ratio<NL, CPL>(tc, g, errm, y, k1m, h);
  if (g.j == 0) {
    double xn[4];
    y_to_state<MODEL>(ynew, xn);
#pragma unroll
    for (int c = 0; c < 4; ++c) d_xnew[c * n + i] = xn[c];
    d_err[i] = r;
  }
#pragma unroll
  for (int st = 0; st < 7; ++st)
#pragma unroll
    for (int c = 0; c < CPL; ++c) d_k[((long long)st * 4 + (c * NL + g.j)) * n + i] = kall_m[st * CPL + c];
}

template <int MODEL, bool SCRIPT>
static catapult_status prepare(int* per_sm) {
  using MT = ModelTraits<MODEL>;
  CATAPULT_CUDA_TRY(cudaFuncSetAttribute(trace_kernel<MODEL, SCRIPT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)MT::SMEM_BYTES));
  CATAPULT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, trace_kernel<MODEL, SCRIPT>, MT::NT,
                                                                  MT::SMEM_BYTES));
  if (*per_sm < 1) {
    set_error("the tracer kernel does not fit on this device (registers / shared memory)");
    return CATAPULT_ECUDA;
  }
  return CATAPULT_OK;
}

template <int MODEL, bool SCRIPT>
static catapult_status shape_for(int64_t n, int* blocks, int* threads) {
  using MT = ModelTraits<MODEL>;
  int dev = 0, sms = 0, per_sm = 0;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  CATAPULT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  catapult_status st = prepare<MODEL, SCRIPT>(&per_sm);
  if (st != CATAPULT_OK) return st;
  const long long resident = (long long)sms * per_sm;  // persistent: a multiple of the SM count
  const long long per_block = MT::NT / MT::NL;         // particles in flight per block
  long long want = (n + per_block - 1) / per_block;
  if (want < 1) want = 1;
  *blocks = (int)(want < resident ? want : resident);
  *threads = MT::NT;
  return CATAPULT_OK;
}

catapult_status trace_launch_shape(int model, int64_t n, int* blocks, int* threads) {
  switch (model) {
    case MODEL_BOOZER_VAC: return shape_for<MODEL_BOOZER_VAC, false>(n, blocks, threads);
    case MODEL_BOOZER_SAW: return shape_for<MODEL_BOOZER_SAW, false>(n, blocks, threads);
    default: return shape_for<MODEL_CART, false>(n, blocks, threads);
  }
}

template <int MODEL, bool SCRIPT>
static catapult_status launch_one(const TraceConst& tc, const TraceArgs& a, cudaStream_t s) {
  using MT = ModelTraits<MODEL>;
  int blocks = 0, threads = 0;
  catapult_status st = shape_for<MODEL, SCRIPT>(a.n, &blocks, &threads);
  if (st != CATAPULT_OK) return st;
  trace_kernel<MODEL, SCRIPT><<<blocks, threads, MT::SMEM_BYTES, s>>>(tc, a);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

catapult_status launch_trace(const TraceConst& tc, const TraceArgs& a, int model, cudaStream_t s) {
  if (a.n == 0) return CATAPULT_OK;
  switch (model) {
    case MODEL_BOOZER_VAC: return launch_one<MODEL_BOOZER_VAC, false>(tc, a, s);
    case MODEL_BOOZER_SAW: return launch_one<MODEL_BOOZER_SAW, false>(tc, a, s);
    default: return launch_one<MODEL_CART, false>(tc, a, s);
  }
}

catapult_status launch_trace_scripted(const TraceConst& tc, const TraceArgs& a, int model, cudaStream_t s) {
  if (a.n == 0) return CATAPULT_OK;
  switch (model) {
    case MODEL_BOOZER_VAC: return launch_one<MODEL_BOOZER_VAC, true>(tc, a, s);
    case MODEL_BOOZER_SAW: return launch_one<MODEL_BOOZER_SAW, true>(tc, a, s);
    default: return launch_one<MODEL_CART, true>(tc, a, s);
  }
}

template <int MODEL>
static catapult_status step_once_one(const TraceConst& tc, int64_t n, const double* d_x, const double* d_t,
                                     const double* d_h, double* d_xnew, double* d_err, double* d_k, cudaStream_t s) {
  using MT = ModelTraits<MODEL>;
  CATAPULT_CUDA_TRY(cudaFuncSetAttribute(step_once_kernel<MODEL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)MT::SMEM_BYTES));
  const long long per_block = MT::NT / MT::NL;
  const int blocks = (int)((n + per_block - 1) / per_block);
  step_once_kernel<MODEL><<<blocks, MT::NT, MT::SMEM_BYTES, s>>>(tc, n, d_x, d_t, d_h, d_xnew, d_err, d_k);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

catapult_status launch_step_once(const TraceConst& tc, int model, int64_t n, const double* d_x, const double* d_t,
                                 const double* d_h, double* d_xnew, double* d_err, double* d_k, cudaStream_t s) {
  if (n == 0) return CATAPULT_OK;
  switch (model) {
    case MODEL_BOOZER_VAC: return step_once_one<MODEL_BOOZER_VAC>(tc, n, d_x, d_t, d_h, d_xnew, d_err, d_k, s);
    case MODEL_BOOZER_SAW: return step_once_one<MODEL_BOOZER_SAW>(tc, n, d_x, d_t, d_h, d_xnew, d_err, d_k, s);
    default: return step_once_one<MODEL_CART>(tc, n, d_x, d_t, d_h, d_xnew, d_err, d_k, s);
  }
}

}  // namespace catapult
