// Persistent fp64 DP5 guiding-centre tracer: warp-specialised, pipelined along the interpolation axes.  This
// kernel serves the cylindrical model (7 tabulated quantities, 3.5 KiB of coefficients per cell); the Boozer models
// (4 quantities) are served by the warp-pair kernel of tracer_pair.cu, which launch_trace() dispatches to.
//
// What is computed is PAPER.md:57-61 (DESIGN.md sections 1-2); the launch shape is this library's own.
//
// A block serves 32 particle slots with NQ + 1 warps (NQ = tabulated quantities):
//   * the SCALAR warp: lane l owns particle slot l -- state, DP5 stage states, cell locate, the guiding-centre
//     physics, error norm, controller, stop test and refill.  One warp instruction advances 32 particles.
//   * NQ CONTRACTION warps: lane l of warp q owns the 64 tricubic coefficients of quantity q of slot l's
//     current cell, on chip (half in registers, half in a private conflict-free run of shared memory),
//     re-fetched from the cell-major table only when the slot's cell changes.
//
// One right-hand-side evaluation ("round") is a two-sided pipeline instead of a ping-pong.  The three local
// coordinates of a stage point do not become known at the same time: the FIRST (zeta / Z) is a state variable,
// the SECOND (s / R) needs a square root, the LAST (theta / phi) an arctangent -- the longest dependent chain of
// the scalar warp.  So the scalar warp publishes (wFIRST, wSECOND) as soon as it has them (barrier A) and goes on
// with the arctangent, the wave terms and the cell index, while the contraction warps contract their 64
// coefficients along FIRST and SECOND (60 of the 63 FMA) on the cell they hold and hand back the four plane
// values P_0..P_3 of every quantity (barrier D); the scalar warp finishes with three FMA per quantity in wLAST.
// The contraction therefore runs entirely in the shadow of the scalar warp's own chain.  The cell a contraction
// lane holds at barrier A is the scalar warp's guess from the round before (fp32 straight-line extrapolation
// along the attempted step, published at barrier G; after the accept/reject decision at barrier G2), fetched
// while the scalar warp works; when the located cell turns out to differ (rare), the lane is told to redo the
// contraction with the right cell (barrier D2).  The contraction warps also accumulate, one state component
// each, the stage partial sums sum_j a_ij k_j and the error-estimate sums, off the scalar warp's critical path.
#include "tracer_common.cuh"

namespace catapult {



template <int MODEL>
struct TraceTraits {
  // this file serves the cylindrical model only (launch_trace below); the Boozer models, the wave included, are
  // tracer_pair.cu's.  The MODEL parameter stays because eval_physics / is_lost / AxisRoles are shared templates.
  static_assert(MODEL == MODEL_CART, "tracer.cu is instantiated for the cylindrical model only");
  static constexpr bool CART = (MODEL == MODEL_CART);
  static constexpr int NQ = CART ? CATAPULT_NQUANT_CYL : CATAPULT_NQUANT_BOOZER;
  static constexpr int NT = 32 * (NQ + 1);   // threads per block
  static constexpr int NCT = 32 * NQ;        // contraction threads per block
  static constexpr int MINB = CART ? 2 : 4;  // resident blocks per SM
  // A contraction thread keeps the first 32 stored coefficients of its (cell, quantity) block (LAST-power 0, 1:
  // gc_device.cuh) in registers and the other 32 in a private run of shared memory: 256 bytes + 16 bytes of
  // padding, so that the 8 lanes of a quarter warp reading 16 bytes each at the same offset of their runs hit 8
  // different 16-byte bank groups.
  static constexpr int STRIP = 272;
  // shared-memory layout (bytes)
  static constexpr size_t OFF_COEF = 0;                               // [NCT] runs of STRIP bytes
  static constexpr size_t OFF_MBAR = OFF_COEF + (size_t)STRIP * NCT;   // uint64 [NCT]: one mbarrier per thread
  static constexpr size_t OFF_PART = OFF_MBAR + 8 * NCT;              // double2 [NQ][2][32]: plane values P_0..P_3
  static constexpr size_t OFF_KS = OFF_PART + (size_t)NQ * 2 * 32 * 16;  // double [7][4][32]: stage derivatives
  static constexpr size_t OFF_W = OFF_KS + 7 * 4 * 32 * 8;            // double [2][32]: wFIRST, wSECOND
  static constexpr size_t OFF_P = OFF_W + 2 * 32 * 8;                 // double [4][32]: stage partial sums
  static constexpr size_t OFF_ERR = OFF_P + 4 * 32 * 8;               // double [8][32]: error sums, 1/denominators
  static constexpr size_t OFF_Y = OFF_ERR + 8 * 32 * 8;               // double [6][32]: y at the step's start, h, dt
  static constexpr size_t OFF_G = OFF_Y + 6 * 32 * 8;                 // int2 [2][32]: (redo cell, next cell) by round parity
  static constexpr size_t OFF_G2 = OFF_G + 2 * 32 * 8;                // int [32]: next cell after the accept/reject decision
  static constexpr size_t OFF_REQ = OFF_G2 + 32 * 4;                  // int [32]: request word
  static constexpr size_t OFF_BASE = OFF_REQ + 32 * 4;                // float [3][32]: start point of the attempt (cell units)
  static constexpr size_t OFF_COLD = OFF_BASE + 3 * 32 * 4;           // per-lane bookkeeping: 7 x int64[32] + 8 x int32[32]
  static constexpr size_t SMEM_BYTES = OFF_COLD + 7 * 256 + 8 * 128;
};

// named barriers (0 is __syncthreads')
constexpr int BAR_A = 1, BAR_D = 2, BAR_G = 3 /* and 4: by round parity */, BAR_D2 = 5, BAR_G2 = 6, BAR_P = 7;
constexpr int NT_P = 32 * 5;  // barrier P: the scalar warp and the four contraction warps that own a state component

__device__ __forceinline__ void bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}


// ---- contraction warps -----------------------------------------------------------------------------------------
template <int MODEL>
__device__ __forceinline__ void contraction_warp(const TraceConst& tc, unsigned char* smem, int q, int lane) {
  using TT = TraceTraits<MODEL>;
  constexpr int NQ = TT::NQ, NT = TT::NT;
  const unsigned FULL = 0xffffffffu;
  const double* __restrict__ table = tc.f.table;
  double reg[32];  // rows (a, b), a = 0, 1: reg[(a*4 + b)*4 + c]
  unsigned char* strip = smem + TT::OFF_COEF + (size_t)(q * 32 + lane) * TT::STRIP;  // rows a = 2, 3
  const unsigned strip_s = smem_u32(strip);
  const unsigned mbar = smem_u32(smem + TT::OFF_MBAR) + 8u * (q * 32 + lane);
  const double* wbuf = reinterpret_cast<const double*>(smem + TT::OFF_W);
  const volatile int* reqbuf = reinterpret_cast<const volatile int*>(smem + TT::OFF_REQ);
  const volatile long long* gbuf = reinterpret_cast<const volatile long long*>(smem + TT::OFF_G);
  const volatile int* g2buf = reinterpret_cast<const volatile int*>(smem + TT::OFF_G2);
  // stage sums: warp q < 4 owns state component q
  const double* ks = reinterpret_cast<const double*>(smem + TT::OFF_KS) + (q & 3) * 32 + lane;  // k_j at ks[j*128]
  double* pbuf = reinterpret_cast<double*>(smem + TT::OFF_P) + (q & 3) * 32 + lane;
  double* errbuf = reinterpret_cast<double*>(smem + TT::OFF_ERR) + (q & 3) * 32 + lane;
  const double* ysm = reinterpret_cast<const double*>(smem + TT::OFF_Y) + lane;
  int cached = -1;
  unsigned phase = 0;    // parity of the mbarrier phase the next wait is for
  bool pending = false;  // a bulk copy into the strip is in flight
  mbar_init(mbar, 1);

  auto wait_strip = [&]() {
    if (pending) {
      mbar_wait(mbar, phase);
      phase ^= 1u;
      pending = false;
    }
  };
  // a cell's 512 contiguous bytes of this lane's quantity: the first half lands in its final registers (eight
  // 256-bit loads), the second half goes global -> shared as ONE bulk asynchronous copy.  Nothing waits here.
  auto issue_loads = [&](int c) {
    const double* src = table + ((long long)c * NQ + q) * 64;
#pragma unroll
    for (int e = 0; e < 32; e += 4) ldg_f64x4(src + e, reg[e], reg[e + 1], reg[e + 2], reg[e + 3]);
    wait_strip();  // an earlier fetch may still be landing in the strip: let it finish first
    mbar_expect_tx(mbar, 256);
    bulk_g2s(strip_s, src + 32, 256, mbar);
    pending = true;
  };
  // P_a = sum_bc C[a][b][c] wS^b wF^c for a = 0..3 (horner_plane of gc_device.cuh: same operations, same order).
  // The shared half streams through two 4-register row buffers, one row in flight while the other is worked
  // on, rows b = 3, 2, 1, 0 of a plane in turn (Horner in wS); the register half fills the gaps.
  const unsigned part_s = smem_u32(smem + TT::OFF_PART) + ((q * 2) * 32 + lane) * 16;
  auto contract = [&](double wF, double wS) {
    double va[4], vb[4];
    lds_row(strip_s + 3 * 32, va);  // plane 2, row 3
    lds_row(strip_s + 2 * 32, vb);  // plane 2, row 2
    auto plane_reg = [&](int a) {
      double row[4];
#pragma unroll
      for (int b = 0; b < 4; ++b) row[b] = reg[(a * 4 + b) * 4 + 3];
#pragma unroll
      for (int c = 2; c >= 0; --c)
#pragma unroll
        for (int b = 0; b < 4; ++b) row[b] = fma(row[b], wF, reg[(a * 4 + b) * 4 + c]);
      return horner_row(row[0], row[1], row[2], row[3], wS);
    };
    const double P0 = plane_reg(0);
    double acc = horner_row(va[0], va[1], va[2], va[3], wF);
    lds_row(strip_s + 1 * 32, va);  // plane 2, row 1
    acc = fma(acc, wS, horner_row(vb[0], vb[1], vb[2], vb[3], wF));
    lds_row(strip_s + 0 * 32, vb);  // plane 2, row 0
    const double P1 = plane_reg(1);
    sts_f64x2(part_s, P0, P1);
    acc = fma(acc, wS, horner_row(va[0], va[1], va[2], va[3], wF));
    lds_row(strip_s + 7 * 32, va);  // plane 3, row 3
    const double P2 = fma(acc, wS, horner_row(vb[0], vb[1], vb[2], vb[3], wF));
    lds_row(strip_s + 6 * 32, vb);  // plane 3, row 2
    acc = horner_row(va[0], va[1], va[2], va[3], wF);
    lds_row(strip_s + 5 * 32, va);  // plane 3, row 1
    acc = fma(acc, wS, horner_row(vb[0], vb[1], vb[2], vb[3], wF));
    lds_row(strip_s + 4 * 32, vb);  // plane 3, row 0
    acc = fma(acc, wS, horner_row(va[0], va[1], va[2], va[3], wF));
    const double P3 = fma(acc, wS, horner_row(vb[0], vb[1], vb[2], vb[3], wF));
    sts_f64x2(part_s + 32 * 16, P2, P3);
  };

  for (;;) {
    bar_sync(BAR_A, NT);
    const int rq = reqbuf[lane];
    if (rq & REQ_QUIT) {  // block-uniform
      wait_strip();    // nothing may still be landing in shared memory when the block retires
      break;
    }
    const bool active = rq & 1;
    const int kind = (rq >> 1) & 7;  // block-uniform
    const int rpar = (rq >> 6) & 1;
    const double wF = wbuf[lane], wS = wbuf[32 + lane];
    if (active) {
      wait_strip();
      contract(wF, wS);
    }
    __syncwarp();
    bar_arrive(BAR_D, NT);
    // ---- stage algebra of state component q: what the next round's stage state needs of the
    // derivatives known so far; in the last round of an attempt everything of Eq. 4 that does not
    // need the last derivative: c = (1,1,1,v_total), state and derivative at the start of the step
    if (q < 4 && kind < KIND_START) {
      switch (kind) {
        case 0: pbuf[0] = stage_partial<1>(ks); break;
        case 1: pbuf[0] = stage_partial<2>(ks); break;
        case 2: pbuf[0] = stage_partial<3>(ks); break;
        case 3: pbuf[0] = stage_partial<4>(ks); break;
        case 4: pbuf[0] = stage_partial<5>(ks); break;
        default: {
          double k[6];
#pragma unroll
          for (int j = 0; j < 6; ++j) k[j] = ks[j * 128];
          double e = 0.0;
#pragma unroll
          for (int j = 0; j < 6; ++j)
            if (j != 1) e = fma(DP_E[j], k[j], e);
          errbuf[0] = e;
          const double sc = (q == 3) ? tc.atol * tc.vtot : tc.atol;
          const double ah = fabs(ysm[4 * 32]);
          errbuf[4 * 32] = fm::rcp(fma(tc.rtol, fma(ah, fabs(k[0]), fabs(ysm[q * 32])), sc));
        }
      }
      __syncwarp();
      bar_arrive(BAR_P, NT_P);
    }
    // ---- the scalar warp has located the point: a wrong cell is redone; then the guessed cell of the next
    // point is fetched while the scalar warp works on
    bar_sync(BAR_G + rpar, NT);
    const long long g = gbuf[rpar * 32 + lane];
    const int redo_cell = (int)g, next_cell = (int)(g >> 32);
    const bool redo = active && redo_cell >= 0;
    if (__any_sync(FULL, redo)) {  // the same answer in every warp of the block
      if (redo) {
        issue_loads(redo_cell);
        cached = redo_cell;
        wait_strip();
        contract(wF, wS);
      }
      __syncwarp();
      bar_arrive(BAR_D2, NT);
    }
    if (active && next_cell >= 0 && next_cell != cached) {
      issue_loads(next_cell);
      cached = next_cell;
    }
    if (kind == 5) {  // end of an attempt: the first point of the next one depends on the accept/reject decision
      bar_sync(BAR_G2, NT);
      const int t2 = g2buf[lane];
      if (active && t2 >= 0 && t2 != cached) {
        issue_loads(t2);
        cached = t2;
      }
    }
  }
}

// ---- scalar warp ---------------------------------------------------------------------------------------------

struct ScalarRegs {   // what the scalar warp carries from round to round besides the particle state
  int rpar;           // parity of the round (the guess buffer and its barrier are double-buffered by it)
  int held;           // the cell this slot's contraction lanes hold (or are fetching)
  unsigned n_load;    // cells fetched for this slot ...
  unsigned n_block;   // ... of which after the point had been located (the guess missed)
};

// Loss time inside the crossing step for the cylindrical model (include/catapult.h loss_time_mode 1, S5b;
// the loss test is a sign change of the INTERPOLATED level function, column 6).  Same construction as
// loss_refine_boozer (gc_device.cuh): the cubic Hermite interpolant through the step's end states and end derivatives,
// 48 bisections from [0, 1] on "level(y(theta)) >= psi_edge", the smallest theta observed beyond the boundary returned
// and y(theta) left in yb.  The level at an interior point needs a table evaluation; the lost lane does it by itself
// straight from the table (locate + the 63-FMA Horner form every user of the table follows, as catapult_field_eval),
// not through the contraction warps: it runs once per lost particle, out of line, so that the stepping loop keeps its
// registers.
__device__ __noinline__ double loss_refine_cart(const FieldConst& f, const double ya[4], const double ka[4],
                                                double yb[4], const double kb[4], double h) {
  using AX = AxisRoles<false>;
  double lo = 0.0, hi = 1.0, ym[4];
#pragma unroll 1
  for (int it = 0; it < 48; ++it) {
    const double mid = 0.5 * (lo + hi);
    hermite_state(ya, ka, yb, kb, h, mid, ym);
    double R, invR, w[3];
    fm::sqrt_rsqrt(fma(ym[0], ym[0], ym[1] * ym[1]), R, invR);
    const int cell = locate<false>(f, R, ym[2], fm::atan2(ym[1], ym[0]), w);
    const double* src = f.table + ((long long)cell * CATAPULT_NQUANT_CYL + (CATAPULT_NQUANT_CYL - 1)) * 64;
    const double level = horner64(
        [&](int e, double& f0, double& f1, double& f2, double& f3) { ldg_f64x4(src + e, f0, f1, f2, f3); },
        w[AX::LAST], w[AX::SECOND], w[AX::FIRST]);
    if (level >= f.psi0) hi = mid;
    else lo = mid;
  }
  hermite_state(ya, ka, yb, kb, h, hi, ym);
#pragma unroll
  for (int i = 0; i < 4; ++i) yb[i] = ym[i];
  return hi;
}

// One lock-step right-hand-side evaluation of the scalar warp at the point (tr, X): see the top of this file.
// Lanes with act = false publish a request nobody serves.  ratio >= 0: the next point is expected at
// X + ratio (X - start of the attempt) and its cell is fetched ahead.  All 32 lanes must call this.
template <int MODEL>
__device__ __forceinline__ void scalar_round(const TraceConst& tc, unsigned char* smem, int lane, bool act, int kind,
                                             ScalarRegs& sr, double tr, const double X[4], double mu, float ratio,
                                             float pos[3], double dy[4], double& modB, double& level) {
  using TT = TraceTraits<MODEL>;
  constexpr bool BZ = (MODEL != MODEL_CART);
  using AX = AxisRoles<BZ>;
  constexpr int NT = TT::NT;
  const unsigned FULL = 0xffffffffu;
  const FieldConst& f = tc.f;
  double* wbuf = reinterpret_cast<double*>(smem + TT::OFF_W);
  int* reqbuf = reinterpret_cast<int*>(smem + TT::OFF_REQ);
  int2* gbuf = reinterpret_cast<int2*>(smem + TT::OFF_G);
  const float* basebuf = reinterpret_cast<const float*>(smem + TT::OFF_BASE);
  EvalGeo g;
  int ci[3];
  double wF, wS, wL;
  // ---- the two coordinates that are known early
  const double r2 = fma(X[0], X[0], X[1] * X[1]);
  fm::sqrt_rsqrt(r2, g.a, g.inva);
  {
    double xr = X[2] - f.lo[AX::FIRST];
    if (BZ) xr = wrap_periodic(xr, f.span[AX::FIRST], f.invspan[AX::FIRST]);
    ci[AX::FIRST] = cell_and_w(xr, f.invh[AX::FIRST], f.k[AX::FIRST], wF, pos[AX::FIRST]);
  }
  ci[AX::SECOND] = cell_and_w(g.a - f.lo[AX::SECOND], f.invh[AX::SECOND], f.k[AX::SECOND], wS, pos[AX::SECOND]);
  wbuf[lane] = wF;
  wbuf[32 + lane] = wS;
  sr.rpar ^= 1;
  reqbuf[lane] = (act ? 1 : 0) | (kind << 1) | (sr.rpar << 6);
  __syncwarp();
  bar_arrive(BAR_A, NT);
  // ---- in the shadow of the arctangent: the unit vector
  g.ca = (BZ && !(g.a > 0.0)) ? 1.0 : X[0] * g.inva;
  g.sa = X[1] * g.inva;
  // ---- the last coordinate and the cell
  {
    const double ang = fm::atan2(X[1], X[0]);
    const double xr = wrap_periodic(ang - f.lo[AX::LAST], f.span[AX::LAST], f.invspan[AX::LAST]);
    ci[AX::LAST] = cell_and_w(xr, f.invh[AX::LAST], f.k[AX::LAST], wL, pos[AX::LAST]);
  }
  const int cell = flat_cell(f, ci[0], ci[1], ci[2]);
  const bool bad = act && cell != sr.held;  // the contraction ran on another cell's coefficients: redo
  int target = -1;
  if (act && ratio >= 0.f) {
    const float base[3] = {basebuf[lane], basebuf[32 + lane], basebuf[64 + lane]};
    target = guess_cell<MODEL>(f, pos, base, ratio);
  }
  gbuf[sr.rpar * 32 + lane] = make_int2(bad ? cell : -1, target);
  if (act) {
    const int now = bad ? cell : sr.held;
    const int next = target >= 0 ? target : now;
    sr.n_block += bad;
    sr.n_load += (unsigned)bad + (unsigned)(next != now);
    sr.held = next;
  }
  __syncwarp();
  bar_arrive(BAR_G + sr.rpar, NT);
  const bool anybad = __any_sync(FULL, bad);
  bar_sync(BAR_D, NT);
  if (anybad) bar_sync(BAR_D2, NT);
  // ---- plane values -> field values (the last three FMA of horner64), then the right-hand side
  const double2* part = reinterpret_cast<const double2*>(smem + TT::OFF_PART) + lane;
  double fv[TT::NQ];
#pragma unroll
  for (int q = 0; q < TT::NQ; ++q) {
    const double2 p01 = part[(q * 2) * 32], p23 = part[(q * 2 + 1) * 32];
    fv[q] = horner_row(p01.x, p01.y, p23.x, p23.y, wL);
  }
  eval_physics<MODEL>(tc, X, mu, g, fv, dy, modB, level);
}

template <int MODEL, int MODE>
__global__ void __launch_bounds__(TraceTraits<MODEL>::NT, TraceTraits<MODEL>::MINB)
trace_kernel(const __grid_constant__ TraceConst tc, const __grid_constant__ TraceArgs a) {
  using TT = TraceTraits<MODEL>;
  extern __shared__ __align__(16) unsigned char smem[];
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  if (warp < TT::NQ) {
    contraction_warp<MODEL>(tc, smem, warp, lane);
    return;
  }

  // ---- scalar warp ------------------------------------------------------------------------------------
  const unsigned FULL = 0xffffffffu;
  const long long n = a.n;
  // DESIGN.md S3: default step lengths (Boozer: L = |G| / |B|(node 0), read from the device scalar the field
  // build left; the cylindrical default is resolved on the host)
  double dtmax = tc.dtmax, dt0 = tc.dt0;
  if (!(dtmax > 0.0)) {
    const double L = __ddiv_rn(fabs(tc.f.G), fabs(*tc.f.node0));
    dtmax = __ddiv_rn(__dmul_rn(0.5 * 3.14159265358979323846, L), tc.vtot);
    dt0 = dt0 > 0.0 ? dt0 : __dmul_rn(1e-3, dtmax);
    dt0 = dt0 > dtmax ? dtmax : dt0;
  }
  double* ks = reinterpret_cast<double*>(smem + TT::OFF_KS) + lane;    // k_j component c at ks[(j*4+c)*32]
  double* ysm = reinterpret_cast<double*>(smem + TT::OFF_Y) + lane;    // y_c of the step's start at ysm[c*32]
  double& hsm = ysm[4 * 32];                                          // length of the attempted step
  double& dt = ysm[5 * 32];                                           // the controller's step length
  const double* pbuf = reinterpret_cast<const double*>(smem + TT::OFF_P) + lane;
  const double* errbuf = reinterpret_cast<const double*>(smem + TT::OFF_ERR) + lane;  // [c]: sum, [4 + c]: 1/denominator
  float* basebuf = reinterpret_cast<float*>(smem + TT::OFF_BASE) + lane;
  int* g2buf = reinterpret_cast<int*>(smem + TT::OFF_G2);
  dt = 0.0;
  hsm = 0.0;
  double t = 0.0, mu = 0.0;
  // bookkeeping that is touched once per attempted step or once per particle lives in shared memory
  long long* cold64 = reinterpret_cast<long long*>(smem + TT::OFF_COLD) + lane;
  unsigned* cold32 = reinterpret_cast<unsigned*>(smem + TT::OFF_COLD + 7 * 256) + lane;
  long long& idx = cold64[0 * 32];
  long long& attempts_left = cold64[1 * 32];
  unsigned long long& c_acc = reinterpret_cast<unsigned long long&>(cold64[2 * 32]);
  unsigned long long& c_rej = reinterpret_cast<unsigned long long&>(cold64[3 * 32]);
  unsigned long long& c_eval = reinterpret_cast<unsigned long long&>(cold64[4 * 32]);
  unsigned long long& c_load = reinterpret_cast<unsigned long long&>(cold64[5 * 32]);
  unsigned long long& c_block = reinterpret_cast<unsigned long long&>(cold64[6 * 32]);
  unsigned& nacc = cold32[0 * 32];
  unsigned& nrej = cold32[1 * 32];
  int& consecutive = reinterpret_cast<int&>(cold32[2 * 32]);
  int& step = reinterpret_cast<int&>(cold32[3 * 32]);
  unsigned* c_fin = cold32 + 4 * 32;  // c_fin[s] at c_fin[s * 32]
  idx = -1;
  attempts_left = 0;
  c_acc = c_rej = c_eval = c_load = c_block = 0;
  nacc = nrej = 0;
  consecutive = step = 0;
#pragma unroll
  for (int j = 0; j < 4; ++j) c_fin[j * 32] = 0;
  bool active = false, exhausted = false;
  ScalarRegs sr{0, -1, 0u, 0u};
  unsigned long long rounds = 0;  // warp-uniform

  for (;;) {
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
      double dy0[4], B, level;
      float pos[3];
      scalar_round<MODEL>(tc, smem, lane, fresh, KIND_START, sr, t, y, 0.0, -1.f, pos, dy0, B, level);
      ++rounds;
      if (fresh) {
        ++c_eval;
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
          ++c_fin[CATAPULT_ST_LOST * 32];
        } else if (MODE != MODE_STEP_ONCE && a.init_only) {
          a.t_io[idx] = 0.0;
          a.status[idx] = CATAPULT_ST_REACHED_T;
          a.dt_io[idx] = dt;
          a.mu_io[idx] = mu;
        } else {
          active = true;
        }
      }
      // k1 with the particle's own mu (mu enters the right-hand side linearly; the round is simply repeated:
      // once per particle)
      const bool go = fresh && active;
      if (__any_sync(FULL, go)) {
        scalar_round<MODEL>(tc, smem, lane, go, KIND_START, sr, t, y, mu, -1.f, pos, dy0, B, level);
        ++rounds;
        if (go) {
          ++c_eval;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            ks[c * 32] = dy0[c];
            ysm[c * 32] = y[c];
          }
#pragma unroll
          for (int d = 0; d < 3; ++d) basebuf[d * 32] = pos[d];  // the first attempt is extrapolated from here
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
      double X[4], dy[4], B_, level = 0.0;
      float pos[3];
      hsm = h;
#pragma unroll
      for (int c = 0; c < 4; ++c) dy[c] = ks[c * 32];  // k1 (first-same-as-last, or the start point's derivative)
#pragma unroll 1
      for (int r = 0; r < 6; ++r) {
        // stage state y + h sum_{j<=r} a[r][j] k_j (row 5 = b: the new state); the sum over j < r was
        // accumulated by the contraction warps during the previous round, the newest derivative enters last
        const double ad = DP_A[r][r];
        if (r > 0) bar_sync(BAR_P, NT_P);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const double Pc = r > 0 ? pbuf[c * 32] : 0.0;
          X[c] = fma(h, fma(ad, dy[c], Pc), ysm[c * 32]);
        }
        const float ratio = (MODE == MODE_STEP_ONCE && r == 5) ? -1.f : NEXT_POINT_RATIO[r];
        scalar_round<MODEL>(tc, smem, lane, stepping, r, sr, fma(DP_C[r], h, t), X, mu, ratio, pos, dy, B_, level);
#pragma unroll
        for (int c = 0; c < 4; ++c) ks[((r + 1) * 4 + c) * 32] = dy[c];
      }
      rounds += 6;
      // PAPER.md:85 Eq. 4: the contraction warps left the sums over the first six derivatives and the
      // reciprocal denominators
      bar_sync(BAR_P, NT_P);
      double r = 0.0, chk = 0.0;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const double e = fma(DP_E[6], dy[c], errbuf[c * 32]) * h;
        const double v = fabs(e) * errbuf[(4 + c) * 32];
        chk += v;
        r = fmax(r, v);
      }
      r = (chk == chk) ? r : chk;  // a non-finite component is a rejection
      bool accepted = false;
      double dtn = h;
      if (MODE == MODE_SCRIPT) accepted = true;
      else if (MODE == MODE_ADAPTIVE) dtn = controller(h, r, dtmax, accepted);
      {
        // the decision goes to the contraction warps at once: the cell of the next attempt's first point, a
        // fifth of the next step length beyond the new start point (accepted: the end point; rejected: the old
        // start point)
        int target = -1;
        if (MODE != MODE_STEP_ONCE && stepping) {
          double hn = h;
          if (MODE == MODE_ADAPTIVE) {
            const double tn = accepted ? (clamped ? tc.T : t + h) : t;
            hn = fmin((accepted && clamped) ? dt : dtn, tc.T - tn);
          }
          const float fr = 0.2f * __fdividef((float)hn, (float)h);
          const float base[3] = {basebuf[0], basebuf[32], basebuf[64]};
          target = guess_cell<MODEL>(tc.f, pos, base, accepted ? fr : fr - 1.0f);
          sr.n_load += (unsigned)(target != sr.held);
          sr.held = target;
          if (accepted) {
#pragma unroll
            for (int d = 0; d < 3; ++d) basebuf[d * 32] = pos[d];
          }
        }
        g2buf[lane] = target;
        __syncwarp();
        bar_arrive(BAR_G2, TT::NT);
      }
      if (stepping) {
        c_eval += 6;
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
            for (int c = 0; c < 4; ++c) a.kall[((long long)j * 4 + c) * n + idx] = ks[(j * 4 + c) * 32];
          active = false;
        }
        if (MODE != MODE_STEP_ONCE) {
          if (!accepted) {
            ++nrej;
            dt = dtn;
            if (++consecutive >= tc.max_rej) finish = CATAPULT_ST_STALLED;  // DESIGN.md S6
          } else {
            consecutive = 0;
            ++nacc;
            const bool lost = is_lost<MODEL>(tc, level);
            if (lost && tc.loss_time_mode == 1) {
              // DESIGN.md S5b: the loss time and state inside this step
              const double ya[4] = {ysm[0], ysm[32], ysm[64], ysm[96]};
              const double ka[4] = {ks[0], ks[32], ks[64], ks[96]};
              // copies: only arrays of this rare branch have their address taken, X and dy stay in registers
              double yb[4] = {X[0], X[1], X[2], X[3]};
              const double kb[4] = {dy[0], dy[1], dy[2], dy[3]};
              const double theta = loss_refine_cart(tc.f, ya, ka, yb, kb, h);  // yb <- y(theta)
#pragma unroll
              for (int c = 0; c < 4; ++c) X[c] = yb[c];
              t = __dadd_rn(t, __dmul_rn(theta, h));
            } else {
              t = clamped ? tc.T : t + h;
            }
            if (!clamped) dt = dtn;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              ysm[c * 32] = X[c];
              ks[c * 32] = dy[c];  // first-same-as-last
            }
            // DESIGN.md S5: loss first, then T
            if (lost) finish = CATAPULT_ST_LOST;
            else if (MODE != MODE_SCRIPT && t >= tc.T) finish = CATAPULT_ST_REACHED_T;
          }
        }
      }
    }
    if (active && finish >= 0) {
      double xo[4];
      const double yf[4] = {ysm[0], ysm[32], ysm[64], ysm[96]};
      y_to_state<MODEL>(yf, xo);
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
      c_load += sr.n_load;
      c_block += sr.n_block;
      sr.n_load = sr.n_block = 0;
      ++c_fin[finish * 32];
      active = false;
    }
  }

  // release the contraction warps
  {
    reinterpret_cast<int*>(smem + TT::OFF_REQ)[lane] = REQ_QUIT;
    __syncwarp();
    bar_arrive(BAR_A, TT::NT);
  }

  // ---- statistics: one atomic per warp per counter -----------------------------------------------------
  if (a.counters) {
    unsigned long long v[CATAPULT_NCOUNTERS] = {c_acc,      c_rej,  c_fin[0],           c_fin[32],           c_fin[64],
                                                c_fin[96],  c_eval, c_load + sr.n_load, c_block + sr.n_block, 0};
#pragma unroll
    for (int j = 0; j < CATAPULT_NCOUNTERS - 1; ++j) {
      unsigned long long s = v[j];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
      if (lane == 0 && s) atomicAdd(a.counters + j, s);
    }
    if (lane == 0 && rounds) atomicAdd(a.counters + CATAPULT_NCOUNTERS - 1, rounds);
  }
}

// ---- launchers ---------------------------------------------------------------------------------------------
// Persistent grid: resident blocks per SM x SM count (or fewer when there are fewer particles than slots).  The
// shape of a (model, mode) pair on a device is computed once and cached.
struct LaunchShape {
  int device = -1, resident = 0;
};

template <int MODEL, int MODE>
static catapult_status trace_shape(int64_t n, int* blocks, int* threads) {
  using TT = TraceTraits<MODEL>;
  static thread_local LaunchShape cache;
  int dev = 0;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  if (cache.device != dev) {
    int sms = 0, per_sm = 0;
    CATAPULT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CATAPULT_CUDA_TRY(cudaFuncSetAttribute(trace_kernel<MODEL, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)TT::SMEM_BYTES));
    CATAPULT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_kernel<MODEL, MODE>, TT::NT,
                                                                    TT::SMEM_BYTES));
    if (per_sm < 1) {
      set_error("the tracer kernel does not fit on this device (registers / shared memory)");
      return CATAPULT_ECUDA;
    }
    cache.device = dev;
    cache.resident = sms * per_sm;  // a multiple of the SM count
  }
  long long want = (n + 31) / 32;
  if (want < 1) want = 1;
  *blocks = (int)(want < cache.resident ? want : cache.resident);
  *threads = TT::NT;
  return CATAPULT_OK;
}

template <int MODEL, int MODE>
static catapult_status trace_launch(const TraceConst& tc, const TraceArgs& a, cudaStream_t s) {
  using TT = TraceTraits<MODEL>;
  int blocks = 0, threads = 0;
  catapult_status st = trace_shape<MODEL, MODE>(a.n, &blocks, &threads);
  if (st != CATAPULT_OK) return st;
  trace_kernel<MODEL, MODE><<<blocks, threads, TT::SMEM_BYTES, s>>>(tc, a);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

template <int MODE>
static catapult_status trace_dispatch(const TraceConst& tc, const TraceArgs& a, int model, cudaStream_t s) {
  if (a.n == 0) return CATAPULT_OK;
  (void)model;  // the Boozer models are served by tracer_pair.cu
  return trace_launch<MODEL_CART, MODE>(tc, a, s);
}

catapult_status launch_trace(const TraceConst& tc, const TraceArgs& a, int model, int mode, cudaStream_t s) {
  if (model != MODEL_CART) return launch_trace_pair(tc, a, model, mode, s);  // tracer_pair.cu
  switch (mode) {
    case MODE_ADAPTIVE: return trace_dispatch<MODE_ADAPTIVE>(tc, a, model, s);
    case MODE_SCRIPT: return trace_dispatch<MODE_SCRIPT>(tc, a, model, s);
    default: return trace_dispatch<MODE_STEP_ONCE>(tc, a, model, s);
  }
}

catapult_status trace_launch_shape(int model, bool doi, int64_t n, int* blocks, int* threads) {
  if (model != MODEL_CART) return trace_pair_shape(model, doi, n, blocks, threads);
  return trace_shape<MODEL_CART, MODE_ADAPTIVE>(n, blocks, threads);
}

}  // namespace catapult
