// Persistent fp64 DP5 guiding-centre tracer, ONE THREAD PER PARTICLE (Boozer models: 4 tabulated quantities).
//
// What is computed is PAPER.md:57-61 (DESIGN.md sections 1-2); the launch shape is this library's own.
//
// One block of 128 threads per SM, one warp per scheduler, up to 255 registers per thread.  Thread t owns particle
// slot t completely: DP5 stage states, cell locate, the tricubic contraction of all four quantities, the
// guiding-centre physics, error norm, controller, stop test and refill.  Nothing is exchanged between threads, so
// the kernel has no barrier and no hand-off; what keeps a scheduler's FP64 pipe busy is the instruction-level
// parallelism of one thread's own work (4 x 16 independent Horner rows beside the square root / arctangent /
// exponential / sine chains of the same evaluation), not other warps.
//
// The 256 coefficients (2 KiB) of the slot's current cell stay ON CHIP from one evaluation to the next: the first
// LANE_NREG of them in registers, the others in a private conflict-free run of shared memory.  They are re-fetched
// from the cell-major table only when the slot's cell changes: the register part by 256-bit read-only loads straight
// into its final registers, the shared part by ONE bulk asynchronous copy (cp.async.bulk) signalled on a
// thread-private mbarrier.  The fetch is issued one evaluation AHEAD, right after the contraction has used the
// old coefficients for the last time, for the cell an fp32 straight-line extrapolation along the attempted step
// predicts (guess_cell); the evaluation contracts speculatively on the cell it holds while its arctangent is
// still in flight and redoes the contraction in the rare case that the located cell differs.
#include "tracer_common.cuh"

namespace catapult {

#ifndef CATAPULT_LANE_AHEAD
#define CATAPULT_LANE_AHEAD 2
#endif
#ifndef CATAPULT_LANE_NREG
#define CATAPULT_LANE_NREG 72
#endif

struct LaneTraits {
  static constexpr int NQ = CATAPULT_NQUANT_BOOZER;
  static constexpr int NCOEF = NQ * 64;
  static constexpr int NREG = CATAPULT_LANE_NREG;  // coefficients kept in registers (a multiple of 4)
  static constexpr int NSH = NCOEF - NREG;         // coefficients kept in shared memory
  static constexpr int NT = 128;                   // threads per block = particle slots per SM
  // one thread's run of shared memory: NSH doubles + 16 bytes of padding, so that the 8 lanes of a quarter warp
  // reading 16 bytes each at the same offset of their runs hit 8 different 16-byte bank groups (STRIP/16 is odd)
  static constexpr int STRIP = NSH * 8 + 16;
  static_assert(NREG % 4 == 0 && NREG > 0 && NREG < NCOEF, "register part: whole rows");
  static_assert((STRIP / 16) % 2 == 1, "run length must be an odd number of 16-byte groups");
  static constexpr size_t OFF_COEF = 0;                                // [NT] runs of STRIP bytes
  static constexpr size_t OFF_MBAR = OFF_COEF + (size_t)STRIP * NT;    // uint64 [NT]: one mbarrier per thread
  static constexpr size_t OFF_KS = OFF_MBAR + 8 * NT;                  // double [7][4][NT]: stage derivatives
  static constexpr size_t OFF_Y = OFF_KS + (size_t)7 * 4 * NT * 8;     // double [6][NT]: y at the step's start, h, dt
  static constexpr size_t OFF_BASE = OFF_Y + (size_t)6 * NT * 8;       // float [3][NT]: start point of the attempt
  static constexpr size_t OFF_COLD = OFF_BASE + (size_t)3 * NT * 4;    // bookkeeping: 2 x int64[NT] + 5 x int32[NT]
  static constexpr size_t SMEM_BYTES = OFF_COLD + (size_t)2 * 8 * NT + (size_t)5 * 4 * NT;
  static_assert(SMEM_BYTES <= 232448, "more than 227 KB of shared memory per block");
};

// What a thread carries about the cell it holds on chip.
constexpr int REPORT_NO_STATUS = 4;

// What an evaluation accumulates on the side, as zero-padded rows of six coefficients of k_1..k_6: during stage
// point r (0..4) the known part of the next stage state (row r + 1 of the tableau without its last entry), during
// the last one (5) the error sums of Eq. 4 over the first six derivatives, during a start point (6)
// nothing.  A zero coefficient meets a derivative of an earlier attempt: those are kept finite (see the kernel).
static __constant__ double LANE_SUMS[7][6] = {
    {3.0 / 40.0, 0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, 0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, 0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 0},
    {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0, -17253.0 / 339200.0, 22.0 / 525.0},
    {0, 0, 0, 0, 0, 0}};

struct LaneCell {
  unsigned strip_s, mbar;      // this thread's run of shared memory and its mbarrier (shared-window addresses)
  int cached;                  // the cell held (or being fetched); -1: none
  unsigned phase;              // parity of the mbarrier phase the next wait is for
  bool pending;                // a bulk copy into the run is in flight
  unsigned n_load, n_block;    // cells fetched for this slot; ... of which after the point had been located
};

__device__ __forceinline__ void lane_wait(LaneCell& lc) {
  if (lc.pending) {
    mbar_wait(lc.mbar, lc.phase);
    lc.phase ^= 1u;
    lc.pending = false;
  }
}

// Fetch of cell c: the first NREG coefficients land in their final registers (256-bit loads), the others go
// global -> shared as ONE bulk asynchronous copy.  Nothing waits here, except for an earlier copy that is still
// landing in the same run.
__device__ __forceinline__ void lane_fetch(const double* __restrict__ table, LaneCell& lc,
                                           double (&creg)[LaneTraits::NREG], int c) {
  using LT = LaneTraits;
  const double* src = table + (long long)c * LT::NCOEF;
#pragma unroll
  for (int e = 0; e < LT::NREG; e += 4) ldg_f64x4(src + e, creg[e], creg[e + 1], creg[e + 2], creg[e + 3]);
  lane_wait(lc);
  mbar_expect_tx(lc.mbar, LT::NSH * 8);
  bulk_g2s(lc.strip_s, src + LT::NREG, LT::NSH * 8, lc.mbar);
  lc.pending = true;
  lc.cached = c;
}

// Four rows (one of each quantity, same powers of wL and wS) by Horner in wF, interleaved so that four
// independent chains are in flight, then one Horner step in wS of the four planes they belong to.  Written as ONE
// statement in the order the FP64 pipe should see, because neither the compiler's front end (which would gather
// all loads of the evaluation ahead of the arithmetic, a register per loaded value) nor the assembler (which keeps
// close to the order it is given) interleaves dependent chains by itself.  FIRST: the rows open their planes.
template <bool FIRST>
__device__ __forceinline__ void quad_rows(const double (&c)[4][4], double wF, double wS, double (&P)[4]) {
  if (FIRST) {
    asm volatile(
        "{\n\t.reg .f64 t0, t1, t2, t3;\n\t"
        "fma.rn.f64 t0, %7, %20, %6;\n\tfma.rn.f64 t1, %11, %20, %10;\n\t"
        "fma.rn.f64 t2, %15, %20, %14;\n\tfma.rn.f64 t3, %19, %20, %18;\n\t"
        "fma.rn.f64 t0, t0, %20, %5;\n\tfma.rn.f64 t1, t1, %20, %9;\n\t"
        "fma.rn.f64 t2, t2, %20, %13;\n\tfma.rn.f64 t3, t3, %20, %17;\n\t"
        "fma.rn.f64 %0, t0, %20, %4;\n\tfma.rn.f64 %1, t1, %20, %8;\n\t"
        "fma.rn.f64 %2, t2, %20, %12;\n\tfma.rn.f64 %3, t3, %20, %16;\n\t}"
        : "=d"(P[0]), "=d"(P[1]), "=d"(P[2]), "=d"(P[3])
        : "d"(c[0][0]), "d"(c[0][1]), "d"(c[0][2]), "d"(c[0][3]), "d"(c[1][0]), "d"(c[1][1]), "d"(c[1][2]),
          "d"(c[1][3]), "d"(c[2][0]), "d"(c[2][1]), "d"(c[2][2]), "d"(c[2][3]), "d"(c[3][0]), "d"(c[3][1]),
          "d"(c[3][2]), "d"(c[3][3]), "d"(wF));
  } else {
    asm volatile(
        "{\n\t.reg .f64 t0, t1, t2, t3;\n\t"
        "fma.rn.f64 t0, %7, %20, %6;\n\tfma.rn.f64 t1, %11, %20, %10;\n\t"
        "fma.rn.f64 t2, %15, %20, %14;\n\tfma.rn.f64 t3, %19, %20, %18;\n\t"
        "fma.rn.f64 t0, t0, %20, %5;\n\tfma.rn.f64 t1, t1, %20, %9;\n\t"
        "fma.rn.f64 t2, t2, %20, %13;\n\tfma.rn.f64 t3, t3, %20, %17;\n\t"
        "fma.rn.f64 t0, t0, %20, %4;\n\tfma.rn.f64 t1, t1, %20, %8;\n\t"
        "fma.rn.f64 t2, t2, %20, %12;\n\tfma.rn.f64 t3, t3, %20, %16;\n\t"
        "fma.rn.f64 %0, %0, %21, t0;\n\tfma.rn.f64 %1, %1, %21, t1;\n\t"
        "fma.rn.f64 %2, %2, %21, t2;\n\tfma.rn.f64 %3, %3, %21, t3;\n\t}"
        : "+d"(P[0]), "+d"(P[1]), "+d"(P[2]), "+d"(P[3])
        : "d"(c[0][0]), "d"(c[0][1]), "d"(c[0][2]), "d"(c[0][3]), "d"(c[1][0]), "d"(c[1][1]), "d"(c[1][2]),
          "d"(c[1][3]), "d"(c[2][0]), "d"(c[2][1]), "d"(c[2][2]), "d"(c[2][3]), "d"(c[3][0]), "d"(c[3][1]),
          "d"(c[3][2]), "d"(c[3][3]), "d"(wF), "d"(wS));
  }
}

// sum_abc C[q][a][b][c] wL^a wS^b wF^c for the four quantities: every row (c) by Horner in wF, the four rows of a
// plane by Horner in wS from b = 3 down, the four planes by Horner in wL from a = 3 down -- the operations and the
// order of horner64 (gc_device.cuh), which every user of the table follows.  The 64 rows are walked with the
// quantity running fastest (quad_rows: 16 quads, plane a = 3 first); the rows of a quad that live in shared
// memory are loaded LANE_AHEAD quads ahead into rotating row buffers.  The walk is cut into steps so that the
// caller can place the scalar chains of the same evaluation between them (the arctangent that gives wL is one of
// them: the plane values need only wF and wS).
struct LaneWalk {
  using LT = LaneTraits;
  static constexpr int AHEAD = CATAPULT_LANE_AHEAD;  // quads between a row's load and its use
  double rb[AHEAD + 1][4][4];
  double P[4][4];  // [a][q]
  static __device__ __forceinline__ constexpr int first_coef(int s, int q) {  // quad s = (a, b) descending
    return q * 64 + ((3 - s / 4) * 4 + (3 - s % 4)) * 4;
  }
  __device__ __forceinline__ void load_quad(unsigned strip_s, int s) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int g = first_coef(s, q);
      if (g >= LT::NREG) lds_row(strip_s + (unsigned)(g - LT::NREG) * 8u, rb[s % (AHEAD + 1)][q]);
    }
  }
  __device__ __forceinline__ void begin(unsigned strip_s) {
#pragma unroll
    for (int s = 0; s < AHEAD; ++s) load_quad(strip_s, s);
  }
  // quads [S0, S1)
  template <int S0, int S1>
  __device__ __forceinline__ void run(const double (&creg)[LT::NREG], unsigned strip_s, double wS, double wF) {
#pragma unroll
    for (int s = S0; s < S1; ++s) {
      if (s + AHEAD < 16) load_quad(strip_s, s + AHEAD);
      double c[4][4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int g = first_coef(s, q);
#pragma unroll
        for (int e = 0; e < 4; ++e) c[q][e] = (g < LT::NREG) ? creg[g < LT::NREG ? g + e : 0] : rb[s % (AHEAD + 1)][q][e];
      }
      if (s % 4 == 0) quad_rows<true>(c, wF, wS, P[3 - s / 4]);
      else quad_rows<false>(c, wF, wS, P[3 - s / 4]);
    }
  }
  __device__ __forceinline__ void finish(double wL, double (&fv)[4]) const {
#pragma unroll
    for (int q = 0; q < 4; ++q) fv[q] = horner_row(P[0][q], P[1][q], P[2][q], P[3][q], wL);
  }
};

// One right-hand-side evaluation of this thread's particle at the point (tr, X).  act = false: the thread has no
// particle in this round (it runs along on whatever it holds and fetches nothing).  ratio >= 0: the next point is
// expected at X + ratio (X - start of the attempt) and its cell is fetched ahead.  S_c = sum_{j < 6} coef[j] k_j,c is
// accumulated on the side (the known part of the next stage state, or of the error estimate; rows of LANE_SUMS).
template <int MODEL>
__device__ __forceinline__ void lane_round(const TraceConst& tc, LaneCell& lc, double (&creg)[LaneTraits::NREG],
                                           bool act, double tr, const double X[4], double mu, float ratio,
                                           const float* basebuf, float pos[3], double dy[4], double& modB,
                                           double& level, const double* coef, const double* ks,
                                           double S[4]) {
  using LT = LaneTraits;
  using AX = AxisRoles<true>;
  const FieldConst& f = tc.f;
  EvalGeo g;
  int ci[3];
  double wF, wS, wL;
  // ---- the two coordinates that are known early
  const double r2 = fma(X[0], X[0], X[1] * X[1]);
  fm::sqrt_rsqrt(r2, g.a, g.inva);
  {
    double xr = X[2] - f.lo[AX::FIRST];
    xr = wrap_periodic(xr, f.span[AX::FIRST], f.invspan[AX::FIRST]);
    ci[AX::FIRST] = cell_and_w(xr, f.invh[AX::FIRST], f.k[AX::FIRST], wF, pos[AX::FIRST]);
  }
  ci[AX::SECOND] = cell_and_w(g.a - f.lo[AX::SECOND], f.invh[AX::SECOND], f.k[AX::SECOND], wS, pos[AX::SECOND]);
  LaneWalk walk;
  int target = -1;
  for (;;) {
    lane_wait(lc);
    // ---- one straight-line block: the contraction along FIRST and SECOND on the cell held (60 of the 63 FMA per
    // quantity) with the arctangent, the wave terms, the stage sums and the next-cell guess placed between its steps
    walk.begin(lc.strip_s);
    walk.run<0, 4>(creg, lc.strip_s, wS, wF);
    {
      const double ang = fm::atan2(X[1], X[0]);
      const double xr = wrap_periodic(ang - f.lo[AX::LAST], f.span[AX::LAST], f.invspan[AX::LAST]);
      ci[AX::LAST] = cell_and_w(xr, f.invh[AX::LAST], f.k[AX::LAST], wL, pos[AX::LAST]);
    }
    walk.run<4, 8>(creg, lc.strip_s, wS, wF);
    g.ca = !(g.a > 0.0) ? 1.0 : X[0] * g.inva;
    g.sa = X[1] * g.inva;
    if (MODEL == MODEL_BOOZER_SAW) {
      const double ds = g.a - tc.saw_s0;
      g.Phihat = tc.saw_Phi0 * fm::exp(-ds * ds * tc.saw_invw2);
      g.dPhihat = g.Phihat * (-2.0 * ds * tc.saw_invw2);
      // sin / cos of m theta - n zeta + omega t by the addition theorem: cos / sin of theta are y0/s, y1/s
      const double beta = fma(-(double)tc.saw_n, X[2], tc.saw_omega * tr);
      double sb, cb, cm, sm;
      fm::sincos(beta, sb, cb);
      unit_power(tc.saw_m, g.ca, g.sa, cm, sm);
      g.sn = fma(sm, cb, cm * sb);
      g.cs = fma(cm, cb, -sm * sb);
    }
    walk.run<8, 12>(creg, lc.strip_s, wS, wF);
#pragma unroll
    for (int c = 0; c < 4; ++c) S[c] = 0.0;
#pragma unroll
    for (int j = 0; j < 6; ++j) {  // coef is a zero-padded row of six: no branch on the number of terms
      const double cj = coef[j];
#pragma unroll
      for (int c = 0; c < 4; ++c) S[c] = fma(cj, ks[(size_t)(j * 4 + c) * LT::NT], S[c]);
    }
    walk.run<12, 16>(creg, lc.strip_s, wS, wF);
    const int cell = flat_cell(f, ci[0], ci[1], ci[2]);
    if (ratio >= 0.f) {
      const float base[3] = {basebuf[0], basebuf[LT::NT], basebuf[2 * LT::NT]};
      target = guess_cell<MODEL>(f, pos, base, ratio);
    }
    if (!(act && cell != lc.cached)) break;
    // the guess of the round before missed (rare): fetch the located cell and contract again
    lane_fetch(f.table, lc, creg, cell);
    ++lc.n_load;
    ++lc.n_block;
  }
  double fv[LT::NQ];
  walk.finish(wL, fv);
  // ---- the cell of the next point, fetched while the rest of this evaluation and the start of the next run
  if (act && target >= 0 && target != lc.cached) {
    lane_fetch(f.table, lc, creg, target);
    ++lc.n_load;
  }
  eval_physics<MODEL>(tc, X, mu, g, fv, dy, modB, level);
}

template <int MODEL, int MODE>
__global__ void __launch_bounds__(LaneTraits::NT, 1)
trace_lane_kernel(const __grid_constant__ TraceConst tc, const __grid_constant__ TraceArgs a, const int lane_cap) {
  using LT = LaneTraits;
  constexpr int NT = LT::NT;
  extern __shared__ __align__(16) unsigned char smem[];
  int tid = threadIdx.x;
  asm volatile("" : "+r"(tid));  // kept in a register: re-reading the special register inside the loop would wait for every load in flight
  const int lane = tid & 31;
  const unsigned FULL = 0xffffffffu;
  const long long n = a.n;

  double creg[LT::NREG];
#pragma unroll
  for (int e = 0; e < LT::NREG; ++e) creg[e] = 0.0;
  LaneCell lc;
  lc.strip_s = smem_u32(smem + LT::OFF_COEF + (size_t)tid * LT::STRIP);
  lc.mbar = smem_u32(smem + LT::OFF_MBAR) + 8u * tid;
  lc.cached = -1;
  lc.phase = 0;
  lc.pending = false;
  lc.n_load = lc.n_block = 0;
  mbar_init(lc.mbar, 1);
  for (int e = 0; e < LT::NSH; ++e) reinterpret_cast<double*>(smem + LT::OFF_COEF + (size_t)tid * LT::STRIP)[e] = 0.0;

  // DESIGN.md S3: default step lengths (L = |G| / |B|(node 0), read from the device scalar the field build left)
  double dtmax = tc.dtmax, dt0 = tc.dt0;
  if (!(dtmax > 0.0)) {
    const double L = __ddiv_rn(fabs(tc.f.G), fabs(*tc.f.node0));
    dtmax = __ddiv_rn(__dmul_rn(0.5 * 3.14159265358979323846, L), tc.vtot);
    dt0 = dt0 > 0.0 ? dt0 : __dmul_rn(1e-3, dtmax);
    dt0 = dt0 > dtmax ? dtmax : dt0;
  }
  double* ks = reinterpret_cast<double*>(smem + LT::OFF_KS) + tid;    // k_j component c at ks[(j*4+c)*NT]
  double* ysm = reinterpret_cast<double*>(smem + LT::OFF_Y) + tid;    // y_c of the step's start at ysm[c*NT]
  double& hsm = ysm[4 * NT];                                         // length of the attempted step
  double& dt = ysm[5 * NT];                                          // the controller's step length
  float* basebuf = reinterpret_cast<float*>(smem + LT::OFF_BASE) + tid;
#pragma unroll 1
  for (int j = 0; j < 28; ++j) ks[j * NT] = 0.0;
#pragma unroll
  for (int j = 0; j < 6; ++j) ysm[j * NT] = 0.0;
  ysm[0] = 1.0;
#pragma unroll
  for (int d = 0; d < 3; ++d) basebuf[d * NT] = 0.f;
  double t = 0.0, mu = 0.0;
  // bookkeeping that is touched once per attempted step or once per particle lives in shared memory
  long long* cold64 = reinterpret_cast<long long*>(smem + LT::OFF_COLD) + tid;
  unsigned* cold32 = reinterpret_cast<unsigned*>(smem + LT::OFF_COLD + (size_t)2 * 8 * NT) + tid;
  long long& idx = cold64[0 * NT];
  long long& attempts_left = cold64[1 * NT];
  unsigned& nacc = cold32[0 * NT];
  unsigned& nrej = cold32[1 * NT];
  int& consecutive = reinterpret_cast<int&>(cold32[2 * NT]);
  int& step = reinterpret_cast<int&>(cold32[3 * NT]);
  unsigned& n_eval = cold32[4 * NT];  // evaluations of the current particle in this call
  idx = -1;
  attempts_left = 0;
  nacc = nrej = n_eval = 0;
  consecutive = step = 0;
  bool active = false;
  int report = -1;  // >= 0: this thread's particle left its slot with this status (REPORT_NO_STATUS: none to count)
  bool exhausted = lane >= lane_cap;  // fewer particles than slots: every warp of the grid takes its share
  unsigned long long rounds = 0;      // warp-uniform

  // statistics of the particles that left their slots: one atomic per warp per counter
  auto flush_reports = [&]() {
    const unsigned reporting = __ballot_sync(FULL, report >= 0);
    if (reporting) {
      if (a.counters) {
        const bool rp = report >= 0;
        unsigned long long v[CATAPULT_NCOUNTERS - 1] = {rp ? nacc : 0u,
                                                        rp ? nrej : 0u,
                                                        report == 0,
                                                        report == 1,
                                                        report == 2,
                                                        report == 3,
                                                        rp ? n_eval : 0u,
                                                        rp ? lc.n_load : 0u,
                                                        rp ? lc.n_block : 0u};
#pragma unroll
        for (int j = 0; j < CATAPULT_NCOUNTERS - 1; ++j) {
          unsigned long long s = v[j];
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
          if (lane == 0 && s) atomicAdd(a.counters + j, s);
        }
      }
      if (report >= 0) {
        lc.n_load = lc.n_block = 0;
        n_eval = 0;
        report = -1;
      }
    }
  };

  for (;;) {
    flush_reports();
    // ---- refill: lanes without a particle pull the next index (one atomic per warp) ------------------
    const bool want = !active && !exhausted;
    const unsigned need = __ballot_sync(FULL, want);
    bool fresh = false;
    double x[4] = {0.0, 0.0, 0.0, 0.0}, y[4] = {1.0, 0.0, 0.0, 0.0};
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
      double dy0[4], B, level, S[4];
      float pos[3];
      lane_round<MODEL>(tc, lc, creg, fresh, t, y, 0.0, -1.f, basebuf, pos, dy0, B, level, LANE_SUMS[6], ks, S);
      ++rounds;
      if (fresh) {
        n_eval = 1;
        nacc = nrej = 0;
        if (MODE != MODE_STEP_ONCE && a.resume) {
          mu = a.mu_io[idx];
          dt = a.dt_io[idx];
        } else {
          mu = (tc.vtot2 - x[3] * x[3]) / (2.0 * B);
          dt = dt0;
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
          report = CATAPULT_ST_LOST;
        } else if (MODE != MODE_STEP_ONCE && a.init_only) {
          a.t_io[idx] = 0.0;
          a.status[idx] = CATAPULT_ST_REACHED_T;
          a.dt_io[idx] = dt;
          a.mu_io[idx] = mu;
          report = REPORT_NO_STATUS;
        } else {
          active = true;
        }
      }
      // k1 with the particle's own mu (mu enters the right-hand side linearly; the round is simply repeated:
      // once per particle)
      const bool go = fresh && active;
      if (__any_sync(FULL, go)) {
        lane_round<MODEL>(tc, lc, creg, go, t, y, mu, -1.f, basebuf, pos, dy0, B, level, LANE_SUMS[6], ks, S);
        ++rounds;
        if (go) {
          ++n_eval;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            ks[c * NT] = dy0[c];
            ysm[c * NT] = y[c];
          }
#pragma unroll
          for (int d = 0; d < 3; ++d) basebuf[d * NT] = pos[d];  // the first attempt is extrapolated from here
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
      double X[4], dy[4], S[4] = {0.0, 0.0, 0.0, 0.0}, B_, level = 0.0;
      float pos[3];
      hsm = h;
#pragma unroll
      for (int c = 0; c < 4; ++c) dy[c] = ks[c * NT];  // k1 (first-same-as-last, or the start point's derivative)
#pragma unroll 1
      for (int r = 0; r < 6; ++r) {
        // stage state y + h sum_{j<=r} a[r][j] k_j (row 5 = b: the new state); the sum over j < r was
        // accumulated during the previous evaluation (S), the newest derivative enters last
        const double ad = DP_A[r][r];
#pragma unroll
        for (int c = 0; c < 4; ++c) X[c] = fma(h, fma(ad, dy[c], S[c]), ysm[c * NT]);
        const float ratio = (MODE == MODE_STEP_ONCE && r == 5) ? -1.f : NEXT_POINT_RATIO[r];
        // on the side: the known part of the next stage state; in the last round the error sums of Eq. 4
        // over the first six derivatives
        lane_round<MODEL>(tc, lc, creg, stepping, fma(DP_C[r], h, t), X, mu, ratio, basebuf, pos, dy, B_, level,
                          LANE_SUMS[r], ks, S);
#pragma unroll
        for (int c = 0; c < 4; ++c) ks[((r + 1) * 4 + c) * NT] = dy[c];
      }
      rounds += 6;
      // PAPER.md:85 Eq. 4 with c = (1,1,1,v_total), state and derivative at the start of the step
      double r = 0.0, chk = 0.0;
      {
        const double ah = fabs(h);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const double sc = (c == 3) ? tc.atol * tc.vtot : tc.atol;
          const double rden = fm::rcp(fma(tc.rtol, fma(ah, fabs(ks[c * NT]), fabs(ysm[c * NT])), sc));
          const double e = fma(DP_E[6], dy[c], S[c]) * h;
          const double v = fabs(e) * rden;
          chk += v;
          r = fmax(r, v);
        }
      }
      r = (chk == chk) ? r : chk;  // a non-finite component is a rejection
      if (MODE != MODE_STEP_ONCE && (!(chk == chk) || fabs(chk) > 1.7e308)) {
        // the derivatives of this attempt will meet zero coefficients in the next one's sums: keep them finite
#pragma unroll 1
        for (int j = 4; j < 28; ++j) ks[j * NT] = 0.0;
      }
      bool accepted = false;
      double dtn = h;
      if (MODE == MODE_SCRIPT) accepted = true;
      else if (MODE == MODE_ADAPTIVE) dtn = controller(h, r, dtmax, accepted);
      if (MODE != MODE_STEP_ONCE && stepping) {
        // the cell of the next attempt's first point, a fifth of the next step length beyond the new start point
        // (accepted: the end point; rejected: the old start point), fetched at once
        double hn = h;
        if (MODE == MODE_ADAPTIVE) {
          const double tn = accepted ? (clamped ? tc.T : t + h) : t;
          hn = fmin((accepted && clamped) ? dt : dtn, tc.T - tn);
        }
        const float fr = 0.2f * __fdividef((float)hn, (float)h);
        const float base[3] = {basebuf[0], basebuf[NT], basebuf[2 * NT]};
        const int target = guess_cell<MODEL>(tc.f, pos, base, accepted ? fr : fr - 1.0f);
        if (target != lc.cached) {
          lane_fetch(tc.f.table, lc, creg, target);
          ++lc.n_load;
        }
        if (accepted) {
#pragma unroll
          for (int d = 0; d < 3; ++d) basebuf[d * NT] = pos[d];
        }
      }
      if (stepping) {
        n_eval += 6;
        if (attempts_left > 0) --attempts_left;
        if (MODE == MODE_SCRIPT) {
          if (a.script_r) a.script_r[(long long)step * n + idx] = r;
          ++step;
        } else if (MODE == MODE_STEP_ONCE) {
          double xn[4];
          y_to_state<MODEL>(X, xn);
#pragma unroll
          for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = xn[c];
          a.script_r[idx] = r;
#pragma unroll
          for (int j = 0; j < 7; ++j)
#pragma unroll
            for (int c = 0; c < 4; ++c) a.kall[((long long)j * 4 + c) * n + idx] = ks[(j * 4 + c) * NT];
          active = false;
          report = REPORT_NO_STATUS;
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
              ysm[c * NT] = X[c];
              ks[c * NT] = dy[c];  // first-same-as-last
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
      const double yf[4] = {ysm[0], ysm[NT], ysm[2 * NT], ysm[3 * NT]};
      y_to_state<MODEL>(yf, xo);
#pragma unroll
      for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = xo[c];
      a.t_io[idx] = t;
      a.status[idx] = finish;
      if (a.dt_io) a.dt_io[idx] = dt;
      if (a.mu_io) a.mu_io[idx] = mu;
      if (a.nacc) a.nacc[idx] = (a.resume ? a.nacc[idx] : 0u) + nacc;
      if (a.nrej) a.nrej[idx] = (a.resume ? a.nrej[idx] : 0u) + nrej;
      report = finish;
      active = false;
    }
  }
  flush_reports();
  lane_wait(lc);  // nothing may still be landing in shared memory when the block retires

  if (a.counters && lane == 0 && rounds) atomicAdd(a.counters + CATAPULT_NCOUNTERS - 1, rounds);
}

// ---- launchers ---------------------------------------------------------------------------------------------
// Persistent grid: one block per SM (or fewer when there are fewer particles than warps could share out).
template <int MODEL, int MODE>
static catapult_status lane_shape(int64_t n, int* blocks, int* threads, int* lane_cap) {
  using LT = LaneTraits;
  static thread_local int cached_device = -1, cached_sms = 0;
  int dev = 0;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  if (cached_device != dev) {
    int sms = 0, per_sm = 0;
    CATAPULT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CATAPULT_CUDA_TRY(cudaFuncSetAttribute(trace_lane_kernel<MODEL, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)LT::SMEM_BYTES));
    CATAPULT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_lane_kernel<MODEL, MODE>, LT::NT,
                                                                    LT::SMEM_BYTES));
    if (per_sm < 1) {
      set_error("the tracer kernel does not fit on this device (registers / shared memory)");
      return CATAPULT_ECUDA;
    }
    cached_device = dev;
    cached_sms = sms;
  }
  long long want = (n + 31) / 32;  // a block is worth starting for 32 particles
  if (want < 1) want = 1;
  const int b = (int)(want < cached_sms ? want : cached_sms);
  // fewer particles than slots: every warp takes an equal share instead of the first warps taking 32 each
  const long long warps = (long long)b * (LT::NT / 32);
  long long cap = (n + warps - 1) / warps;
  *lane_cap = (int)(cap < 1 ? 1 : (cap > 32 ? 32 : cap));
  *blocks = b;
  *threads = LT::NT;
  return CATAPULT_OK;
}

template <int MODEL, int MODE>
static catapult_status lane_launch(const TraceConst& tc, const TraceArgs& a, cudaStream_t s) {
  int blocks = 0, threads = 0, cap = 32;
  catapult_status st = lane_shape<MODEL, MODE>(a.n, &blocks, &threads, &cap);
  if (st != CATAPULT_OK) return st;
  trace_lane_kernel<MODEL, MODE><<<blocks, threads, LaneTraits::SMEM_BYTES, s>>>(tc, a, cap);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

template <int MODE>
static catapult_status lane_dispatch(const TraceConst& tc, const TraceArgs& a, int model, cudaStream_t s) {
  if (a.n == 0) return CATAPULT_OK;
  if (model == MODEL_BOOZER_VAC) return lane_launch<MODEL_BOOZER_VAC, MODE>(tc, a, s);
  return lane_launch<MODEL_BOOZER_SAW, MODE>(tc, a, s);
}

catapult_status launch_trace_lane(const TraceConst& tc, const TraceArgs& a, int model, int mode, cudaStream_t s) {
  switch (mode) {
    case MODE_ADAPTIVE: return lane_dispatch<MODE_ADAPTIVE>(tc, a, model, s);
    case MODE_SCRIPT: return lane_dispatch<MODE_SCRIPT>(tc, a, model, s);
    default: return lane_dispatch<MODE_STEP_ONCE>(tc, a, model, s);
  }
}

catapult_status trace_lane_shape(int model, int64_t n, int* blocks, int* threads) {
  int cap = 0;
  if (model == MODEL_BOOZER_VAC) return lane_shape<MODEL_BOOZER_VAC, MODE_ADAPTIVE>(n, blocks, threads, &cap);
  return lane_shape<MODEL_BOOZER_SAW, MODE_ADAPTIVE>(n, blocks, threads, &cap);
}

}  // namespace catapult
