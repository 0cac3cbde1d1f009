// Persistent fp64 DP5 guiding-centre tracer, warp-specialised ("split") form.
//
// What is computed is PAPER.md:57-61 (DESIGN.md sections 1-2); the launch shape is this library's own.
//
// A block serves 32 particle slots with NQ + 1 warps (NQ = tabulated quantities: 4 Boozer, 7 cylindrical):
//   * the SCALAR warp: lane l owns particle slot l -- state, DP5 stage algebra, cell locate, the
//     guiding-centre physics, error norm, controller, stop test and refill.  Nothing is replicated:
//     one warp instruction advances 32 particles.
//   * NQ CONTRACTION warps: lane l of warp q owns the 64 tricubic coefficients of quantity q of slot l's
//     current cell, on chip (NREG in registers, the rest in a private conflict-free strip of shared
//     memory), re-fetched from the cell-major table only when the slot's cell changes.  Per evaluation it
//     reads the slot's (cell, w) from shared memory, evaluates the 64-coefficient polynomial by nested
//     Horner (63 FMA, gc_device.cuh) and writes one value back.
// The two sides meet through two named barriers per evaluation (bar.arrive / bar.sync producer-consumer
// pairs): the scalar warp publishes (cell, w) and -- while the contraction warps work -- evaluates
// everything that does not need field values (the wave's exp / sincos); then it picks up the NQ values.
// The seven stage derivatives live in shared memory, so the stage loop is rolled (one copy of the
// right-hand side in the instruction stream).
#include "gc_device.cuh"

namespace catapult {

#ifndef CATAPULT_SPLIT_NREG_BOOZER
#define CATAPULT_SPLIT_NREG_BOOZER 32
#endif
#ifndef CATAPULT_SPLIT_NREG_CART
#define CATAPULT_SPLIT_NREG_CART 32
#endif
#ifndef CATAPULT_SPLIT_MINB_BOOZER
#define CATAPULT_SPLIT_MINB_BOOZER 4
#endif
#ifndef CATAPULT_SPLIT_MINB_CART
#define CATAPULT_SPLIT_MINB_CART 2
#endif

constexpr int MODE_ADAPTIVE = 0, MODE_SCRIPT = 1, MODE_STEP_ONCE = 2;

// Dormand-Prince 5(4) tableau for the rolled stage loop (row i = coefficients of the state fed to stage
// i+2; the last row is b: the 7th stage is evaluated at the new state).  PAPER.md:61, ref [10].
__constant__ double DP_A[6][6] = {
    {1.0 / 5.0, 0, 0, 0, 0, 0},
    {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
__constant__ double DP_C[6] = {1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
__constant__ double DP_E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0, -17253.0 / 339200.0,
                               22.0 / 525.0, -1.0 / 40.0};

template <int MODEL>
struct SplitTraits {
  static constexpr bool CART = (MODEL == MODEL_CART);
  static constexpr int NQ = CART ? CATAPULT_NQUANT_CYL : CATAPULT_NQUANT_BOOZER;
  static constexpr int NT = 32 * (NQ + 1);   // threads per block
  static constexpr int NCT = 32 * NQ;        // contraction threads per block
  static constexpr int NREG = CART ? CATAPULT_SPLIT_NREG_CART : CATAPULT_SPLIT_NREG_BOOZER;
  static constexpr int NSH = 64 - NREG;      // coefficients per contraction thread kept in shared memory
  static constexpr int MINB = CART ? CATAPULT_SPLIT_MINB_CART : CATAPULT_SPLIT_MINB_BOOZER;
  static_assert(NREG % 4 == 0 && NREG >= 0 && NREG <= 64, "NREG must be a multiple of 4 in [0,64]");
  // shared-memory layout (bytes)
  static constexpr size_t OFF_COEF = 0;                             // double2 [NSH/2][NCT]
  static constexpr size_t OFF_KS = OFF_COEF + (size_t)NSH * 8 * NCT;  // double [7][4][32]
  static constexpr size_t OFF_U = OFF_KS + 7 * 4 * 32 * 8;          // double [3][32]
  static constexpr size_t OFF_FV = OFF_U + 3 * 32 * 8;              // double [NQ][32]
  static constexpr size_t OFF_CELL = OFF_FV + (size_t)NQ * 32 * 8;  // int    [32]
  static constexpr size_t SMEM_BYTES = OFF_CELL + 32 * 4;
};

constexpr int CELL_NONE = -1;  // slot has nothing to evaluate this round
constexpr int CELL_QUIT = -2;  // the scalar warp is done: contraction warps exit

__device__ __forceinline__ void bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// 16-byte global -> shared copy that bypasses the register file (LDGSTS); completion is per thread
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// ---- contraction warps -----------------------------------------------------------------------------
template <int MODEL>
__device__ __forceinline__ void contraction_warp(const double* __restrict__ table, unsigned char* smem, int q,
                                                 int lane) {
  using ST = SplitTraits<MODEL>;
  constexpr int NQ = ST::NQ, NREG = ST::NREG, NCT = ST::NCT, NT = ST::NT;
  double reg[NREG > 0 ? NREG : 1];
  double2* sl = reinterpret_cast<double2*>(smem + ST::OFF_COEF) + (q * 32 + lane);  // chunk c at sl[c * NCT]
  const double* ubuf = reinterpret_cast<const double*>(smem + ST::OFF_U);
  double* fvbuf = reinterpret_cast<double*>(smem + ST::OFF_FV);
  const volatile int* cellbuf = reinterpret_cast<const volatile int*>(smem + ST::OFF_CELL);
  int cached = CELL_NONE;
  for (;;) {
    bar_sync(1, NT);
    const int c = cellbuf[lane];
    if (c == CELL_QUIT) break;  // warp-uniform
    if (c >= 0) {
      if (c != cached) {
        // a new cell: 512 contiguous bytes of this lane's quantity.  The shared-memory part goes global ->
        // shared without passing through registers (cp.async), the register part lands in its final
        // registers, so all 16 requests are in flight together: one memory latency per cell change.
        const double* src = table + ((long long)c * NQ + q) * 64;
#pragma unroll
        for (int e = NREG; e < 64; e += 2) cp_async16(sl + ((e - NREG) / 2) * NCT, src + e);
#pragma unroll
        for (int e = 0; e < NREG; e += 4) ldg_f64x4(src + e, reg[e], reg[e + 1], reg[e + 2], reg[e + 3]);
        cp_async_wait_all();
        cached = c;
      }
      const double w0 = ubuf[lane], w1 = ubuf[32 + lane], w2 = ubuf[64 + lane];
      const double acc = horner64(
          [&](int e, double& f0, double& f1, double& f2, double& f3) {
            if (e < NREG) {
              f0 = reg[e];
              f1 = reg[e + 1];
              f2 = reg[e + 2];
              f3 = reg[e + 3];
            } else {
              const double2 v01 = sl[((e - NREG) / 2) * NCT];
              const double2 v23 = sl[((e - NREG) / 2 + 1) * NCT];
              f0 = v01.x;
              f1 = v01.y;
              f2 = v23.x;
              f3 = v23.y;
            }
          },
          w0, w1, w2);
      fvbuf[q * 32 + lane] = acc;
    }
    __syncwarp();
    bar_arrive(2, NT);
  }
}

// ---- scalar warp: geometry before the field values are known ------------------------------------------
struct EvalGeo {
  double a, inva, ang;                 // Boozer: s, 1/s, theta;  Cartesian: R, 1/R, phi
  double sn, cs, Phihat, dPhihat;      // wave terms (MODEL_BOOZER_SAW)
};

template <int MODEL>
__device__ __forceinline__ int eval_locate(const TraceConst& tc, const double y[4], double w[3], EvalGeo& g) {
  const double r2 = fma(y[0], y[0], y[1] * y[1]);
  fm::sqrt_rsqrt(r2, g.a, g.inva);
  g.ang = fm::atan2(y[1], y[0]);
  if (MODEL == MODEL_CART) return locate<false>(tc.f, g.a, y[2], g.ang, w);
  return locate<true>(tc.f, g.a, g.ang, y[2], w);
}

// everything of the right-hand side that does not need the interpolated field (overlaps the contraction)
template <int MODEL>
__device__ __forceinline__ void eval_wave(const TraceConst& tc, double t, const double y[4], EvalGeo& g) {
  if (MODEL == MODEL_BOOZER_SAW) {
    const double ds = g.a - tc.saw_s0;
    g.Phihat = tc.saw_Phi0 * fm::exp(-ds * ds * tc.saw_invw2);
    g.dPhihat = g.Phihat * (-2.0 * ds * tc.saw_invw2);
    const double eta = fma((double)tc.saw_m, g.ang, fma(-(double)tc.saw_n, y[2], tc.saw_omega * t));
    fm::sincos(eta, g.sn, g.cs);
  }
}

// DESIGN.md R1-R3 with the interpolated values fv
template <int MODEL>
__device__ __forceinline__ void eval_physics(const TraceConst& tc, const double y[4], double mu, const EvalGeo& g,
                                             const double* fv, double dy[4], double& modB, double& level) {
  const FieldConst& f = tc.f;
  if (MODEL == MODEL_CART) {
    const double cph = y[0] * g.inva, sph = y[1] * g.inva;
    const double BR = fv[0], Bp = fv[1], BZ = fv[2], gR = fv[3], gp = fv[4], gZ = fv[5];
    const double Bx = BR * cph - Bp * sph, By = BR * sph + Bp * cph, Bz = BZ;
    const double gx = gR * cph - gp * sph, gy = gR * sph + gp * cph, gz = gZ;
    const double B2 = fma(BR, BR, fma(Bp, Bp, BZ * BZ));
    double B, invB;
    fm::sqrt_rsqrt(B2, B, invB);
    const double vpar = y[3];
    const double coef = tc.Moq * invB * invB * invB * fma(mu, B, vpar * vpar);
    const double cx = By * gz - Bz * gy, cy = Bz * gx - Bx * gz, cz = Bx * gy - By * gx;
    const double vb = vpar * invB;
    dy[0] = fma(vb, Bx, coef * cx);
    dy[1] = fma(vb, By, coef * cy);
    dy[2] = fma(vb, Bz, coef * cz);
    dy[3] = -mu * invB * fma(Bx, gx, fma(By, gy, Bz * gz));
    modB = B;
    level = fv[6];
  } else {
    const double s = g.a, invs = g.inva;
    const double B = fv[0], B_s = fv[1], B_th = fv[2], B_ze = fv[3];
    const double vpar = y[3];
    const double invB = fm::rcp(B);
    const double W = tc.Moq * fma(vpar * vpar, invB, mu);
    const double iota = fma(f.iota1, s, f.iota0);
    const double B_psi = B_s * f.invpsi0;
    const double vBG = vpar * B * f.invG;
    double sdot, thdot, vdot;
    if (MODEL == MODEL_BOOZER_VAC) {
      sdot = -B_th * W * f.invpsi0;
      thdot = fma(B_psi, W, iota * vBG);
      vdot = -fma(iota, B_th, B_ze) * mu * B * f.invG;
    } else {
      const double mm = (double)tc.saw_m, nn = (double)tc.saw_n;
      const double Phihat = g.Phihat, dPhihat = g.dPhihat, sn = g.sn, cs = g.cs;
      const double Phi = Phihat * sn;
      const double Phi_psi = dPhihat * sn * f.invpsi0;
      const double Phi_th = mm * Phihat * cs;
      const double Phi_ze = -nn * Phihat * cs;
      const double kpar = fma(iota, mm, -nn);
      const double inv_omG = tc.saw_inv_omG;
      const double al_th = -kpar * Phi_th * inv_omG;
      const double al_t = -kpar * Phihat * cs * f.invG;
      const double al_psi = -fma(f.iota1 * mm, Phi, kpar * dPhihat * sn) * inv_omG * f.invpsi0;
      const double psidot = fma(-B_th, W, fma(al_th, B * vpar, -Phi_th));
      sdot = psidot * f.invpsi0;
      const double iag = fma(-al_psi, f.G, iota);  // iota - alpha_psi G
      thdot = fma(B_psi, W, fma(iag * f.invG, vpar * B, Phi_psi));
      const double t1 = tc.M * mu * fma(al_th * B_psi, f.G, fma(B_th, iag, B_ze));
      const double t2 = tc.q * fma(al_t, f.G, fma(al_th * f.G, Phi_psi, fma(iag, Phi_th, Phi_ze)));
      vdot = fma(-(B * f.invG * tc.invM), t1 + t2, vpar * invB * fma(B_th, Phi_psi, -B_psi * Phi_th));
    }
    const double c = (s > 0.0) ? y[0] * invs : 1.0;
    const double sn_ = y[1] * invs;
    dy[0] = fma(sdot, c, -thdot * y[1]);
    dy[1] = fma(sdot, sn_, thdot * y[0]);
    dy[2] = vBG;
    dy[3] = vdot;
    modB = B;
    level = s;
  }
}

// One lock-step evaluation round of the scalar warp: lanes with `on` evaluate the right-hand side at
// (t, y); the others publish CELL_NONE.  Must be called by all 32 lanes.
template <int MODEL>
__device__ __forceinline__ void eval_round(const TraceConst& tc, unsigned char* smem, int lane, bool on, double t,
                                           const double y[4], double mu, double dy[4], double& modB,
                                           double& level) {
  using ST = SplitTraits<MODEL>;
  double* ubuf = reinterpret_cast<double*>(smem + ST::OFF_U);
  const double* fvbuf = reinterpret_cast<const double*>(smem + ST::OFF_FV);
  volatile int* cellbuf = reinterpret_cast<volatile int*>(smem + ST::OFF_CELL);
  EvalGeo g;
  double w[3];
  const int cell = eval_locate<MODEL>(tc, y, w, g);
  ubuf[lane] = w[0];
  ubuf[32 + lane] = w[1];
  ubuf[64 + lane] = w[2];
  cellbuf[lane] = on ? cell : CELL_NONE;
  __syncwarp();
  bar_arrive(1, ST::NT);
  eval_wave<MODEL>(tc, t, y, g);
  bar_sync(2, ST::NT);
  double fv[ST::NQ];
#pragma unroll
  for (int q = 0; q < ST::NQ; ++q) fv[q] = fvbuf[q * 32 + lane];
  eval_physics<MODEL>(tc, y, mu, g, fv, dy, modB, level);
}

template <int MODEL, int MODE>
__global__ void __launch_bounds__(SplitTraits<MODEL>::NT, SplitTraits<MODEL>::MINB)
trace_kernel(const __grid_constant__ TraceConst tc, const __grid_constant__ TraceArgs a) {
  using ST = SplitTraits<MODEL>;
  extern __shared__ __align__(16) unsigned char smem[];
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  if (warp < ST::NQ) {
    contraction_warp<MODEL>(tc.f.table, smem, warp, lane);
    return;
  }

  // ---- scalar warp ------------------------------------------------------------------------------------
  const unsigned FULL = 0xffffffffu;
  const long long n = a.n;
  double* ks = reinterpret_cast<double*>(smem + ST::OFF_KS) + lane;  // k_j component c at ks[(j*4+c)*32]
  double y[4] = {1.0, 0.0, 0.0, 0.0}, t = 0.0, dt = 0.0, mu = 0.0;
  long long idx = -1;
  unsigned nacc = 0, nrej = 0;
  long long attempts_left = 0;
  int consecutive = 0, step = 0;
  bool active = false, exhausted = false;
  unsigned long long c_acc = 0, c_rej = 0, c_eval = 0;
  unsigned c_fin[4] = {0, 0, 0, 0};

  for (;;) {
    // ---- refill: lanes without a particle pull the next index (one atomic per warp) ------------------
    const bool want = !active && !exhausted;
    const unsigned need = __ballot_sync(FULL, want);
    bool fresh = false;
    double x[4] = {0.0, 0.0, 0.0, 0.0};
    if (need) {
      const int leader = __ffs(need) - 1;
      unsigned long long base = 0;
      if (lane == leader) base = atomicAdd(a.queue, (unsigned long long)__popc(need));
      base = __shfl_sync(FULL, base, leader);
      if (want) {
        const long long mine = (long long)base + __popc(need & ((1u << lane) - 1u));
        if (mine >= n) {
          exhausted = true;
        } else {
          idx = mine;
#pragma unroll
          for (int c = 0; c < 4; ++c) x[c] = a.x_in[c * n + idx];
          bool skip = false;
          if (MODE == MODE_STEP_ONCE) {
            t = a.t_io[idx];
          } else if (a.resume) {
            skip = (a.status[idx] != CATAPULT_ST_REACHED_T);
            t = a.t_io[idx];
            if (!(t < tc.T)) skip = true;  // already at (or past) the requested end time
          } else {
            t = 0.0;
          }
          if (!skip) {
            state_to_y<MODEL>(x, y);
            fresh = true;
          }
        }
      }
    }
    if (__any_sync(FULL, fresh)) {
      // the start point's field values give mu and k1
      double dy0[4], B, level;
      eval_round<MODEL>(tc, smem, lane, fresh, t, y, 0.0, dy0, B, level);
      if (fresh) {
        ++c_eval;
        if (MODE != MODE_STEP_ONCE && a.resume) {
          mu = a.mu_io[idx];
          dt = a.dt_io[idx];
        } else {
          mu = (tc.vtot2 - x[3] * x[3]) / (2.0 * B);
          dt = tc.dt0;
        }
        if (MODE != MODE_STEP_ONCE && !a.resume && is_lost<MODEL>(tc, level)) {
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
        } else if (MODE != MODE_STEP_ONCE && a.init_only) {
          a.t_io[idx] = 0.0;
          a.status[idx] = CATAPULT_ST_REACHED_T;
          a.dt_io[idx] = dt;
          a.mu_io[idx] = mu;
        } else {
          active = true;
        }
      }
      // k1 with the particle's own mu: the field values are those of the round above; only the physics
      // is redone (mu enters linearly; the geometry is recomputed from y, cheap and rare)
      if (__any_sync(FULL, fresh && active)) {
        eval_round<MODEL>(tc, smem, lane, fresh && active, t, y, mu, dy0, B, level);
        if (fresh && active) {
          ++c_eval;
#pragma unroll
          for (int c = 0; c < 4; ++c) ks[c * 32] = dy0[c];
          nacc = 0;
          nrej = 0;
          consecutive = 0;
          step = 0;
          attempts_left = tc.max_steps > 0 ? tc.max_steps : -1;
        }
      }
    }
    if (!__any_sync(FULL, active)) {
      if (__all_sync(FULL, exhausted)) break;
      continue;
    }

    // ---- one attempted step for every active lane -------------------------------------------------------
    int finish = -1;
    double h = 0.0;
    bool clamped = false;
    if (active) {
      if (MODE == MODE_SCRIPT) {
        h = (step < a.script_len) ? a.script_h[(long long)step * n + idx] : 0.0;
        if (!(h > 0.0)) finish = CATAPULT_ST_REACHED_T;
      } else if (MODE == MODE_STEP_ONCE) {
        h = a.script_h[idx];
      } else if (attempts_left == 0) {
        finish = CATAPULT_ST_MAXSTEPS;
      } else {
        const double rem = tc.T - t;
        clamped = !(dt < rem);  // the last step lands exactly on T (S4)
        h = clamped ? rem : dt;
      }
    }
    const bool stepping = active && finish < 0;
    if (__any_sync(FULL, stepping)) {
      double ys[4], dy[4], B_, level = 0.0;
#pragma unroll 1
      for (int st = 0; st < 6; ++st) {
        // stage state: y + h sum_j a[st][j] k_j   (row 5 = b: the new state)
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int j = 0; j < 6; ++j) {
          if (j <= st) {
            const double aj = DP_A[st][j];
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = fma(aj, ks[(j * 4 + c) * 32], acc[c]);
          }
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) ys[c] = fma(h, acc[c], y[c]);
        eval_round<MODEL>(tc, smem, lane, stepping, fma(DP_C[st], h, t), ys, mu, dy, B_, level);
#pragma unroll
        for (int c = 0; c < 4; ++c) ks[((st + 1) * 4 + c) * 32] = dy[c];
      }
      if (stepping) {
        c_eval += 6;
        if (attempts_left > 0) --attempts_left;
        // PAPER.md:85 Eq. 4, c = (1,1,1,v_total), state and derivative at the start of the step
        double r = 0.0, chk = 0.0;
        const double ah = fabs(h);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          double e = 0.0;
#pragma unroll
          for (int j = 0; j < 7; ++j)
            if (j != 1) e = fma(DP_E[j], ks[(j * 4 + c) * 32], e);
          e *= h;
          const double sc = (c == 3) ? tc.atol * tc.vtot : tc.atol;
          const double den = fma(tc.rtol, fma(ah, fabs(ks[c * 32]), fabs(y[c])), sc);
          const double v = fabs(e) * fm::rcp(den);
          chk += v;
          r = fmax(r, v);
        }
        r = (chk == chk) ? r : chk;  // a non-finite component is a rejection
        bool accepted;
        double dtn;
        if (MODE == MODE_SCRIPT) {
          if (a.script_r) a.script_r[(long long)step * n + idx] = r;
          ++step;
          accepted = true;
          dtn = h;
        } else if (MODE == MODE_STEP_ONCE) {
          accepted = false;
          dtn = h;
          double xn[4];
          y_to_state<MODEL>(ys, xn);
#pragma unroll
          for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = xn[c];
          a.script_r[idx] = r;
#pragma unroll
          for (int j = 0; j < 7; ++j)
#pragma unroll
            for (int c = 0; c < 4; ++c) a.kall[((long long)j * 4 + c) * n + idx] = ks[(j * 4 + c) * 32];
          active = false;
        } else {
          dtn = controller(h, r, tc.dtmax, accepted);
        }
        if (MODE != MODE_STEP_ONCE) {
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
            for (int c = 0; c < 4; ++c) {
              y[c] = ys[c];
              ks[c * 32] = dy[c];  // first-same-as-last
            }
            // DESIGN.md S5: loss first, then T
            if (is_lost<MODEL>(tc, level)) finish = CATAPULT_ST_LOST;
            else if (MODE != MODE_SCRIPT && t >= tc.T) finish = CATAPULT_ST_REACHED_T;
          }
        }
      }
    }
    if (active && finish >= 0) {
      double xo[4];
      y_to_state<MODEL>(y, xo);
#pragma unroll
      for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = xo[c];
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

  // release the contraction warps
  {
    volatile int* cellbuf = reinterpret_cast<volatile int*>(smem + ST::OFF_CELL);
    cellbuf[lane] = CELL_QUIT;
    __syncwarp();
    bar_arrive(1, ST::NT);
  }

  // ---- statistics: one atomic per warp per counter -----------------------------------------------------
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

// ---- launchers ---------------------------------------------------------------------------------------------
template <int MODEL, int MODE>
static catapult_status split_shape(int64_t n, int* blocks, int* threads) {
  using ST = SplitTraits<MODEL>;
  int dev = 0, sms = 0, per_sm = 0;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  CATAPULT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  CATAPULT_CUDA_TRY(cudaFuncSetAttribute(trace_kernel<MODEL, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)ST::SMEM_BYTES));
  CATAPULT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_kernel<MODEL, MODE>, ST::NT,
                                                                  ST::SMEM_BYTES));
  if (per_sm < 1) {
    set_error("the tracer kernel does not fit on this device (registers / shared memory)");
    return CATAPULT_ECUDA;
  }
  const long long resident = (long long)sms * per_sm;  // persistent: a multiple of the SM count
  long long want = (n + 31) / 32;
  if (want < 1) want = 1;
  *blocks = (int)(want < resident ? want : resident);
  *threads = ST::NT;
  return CATAPULT_OK;
}

template <int MODEL, int MODE>
static catapult_status split_launch(const TraceConst& tc, const TraceArgs& a, cudaStream_t s) {
  using ST = SplitTraits<MODEL>;
  int blocks = 0, threads = 0;
  catapult_status st = split_shape<MODEL, MODE>(a.n, &blocks, &threads);
  if (st != CATAPULT_OK) return st;
  trace_kernel<MODEL, MODE><<<blocks, threads, ST::SMEM_BYTES, s>>>(tc, a);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

template <int MODE>
static catapult_status split_dispatch(const TraceConst& tc, const TraceArgs& a, int model, cudaStream_t s) {
  if (a.n == 0) return CATAPULT_OK;
  switch (model) {
    case MODEL_BOOZER_VAC: return split_launch<MODEL_BOOZER_VAC, MODE>(tc, a, s);
    case MODEL_BOOZER_SAW: return split_launch<MODEL_BOOZER_SAW, MODE>(tc, a, s);
    default: return split_launch<MODEL_CART, MODE>(tc, a, s);
  }
}

catapult_status launch_trace(const TraceConst& tc, const TraceArgs& a, int model, int mode, cudaStream_t s) {
  switch (mode) {
    case MODE_ADAPTIVE: return split_dispatch<MODE_ADAPTIVE>(tc, a, model, s);
    case MODE_SCRIPT: return split_dispatch<MODE_SCRIPT>(tc, a, model, s);
    default: return split_dispatch<MODE_STEP_ONCE>(tc, a, model, s);
  }
}

catapult_status trace_launch_shape(int model, int64_t n, int* blocks, int* threads) {
  switch (model) {
    case MODEL_BOOZER_VAC: return split_shape<MODEL_BOOZER_VAC, MODE_ADAPTIVE>(n, blocks, threads);
    case MODEL_BOOZER_SAW: return split_shape<MODEL_BOOZER_SAW, MODE_ADAPTIVE>(n, blocks, threads);
    default: return split_shape<MODEL_CART, MODE_ADAPTIVE>(n, blocks, threads);
  }
}

}  // namespace catapult
