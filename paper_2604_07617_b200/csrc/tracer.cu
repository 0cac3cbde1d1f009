// Persistent fp64 DP5 guiding-centre tracer, warp-specialised ("split") form.
//
// What is computed is PAPER.md:57-61 (DESIGN.md sections 1-2); the launch shape is this library's own.
//
// A block serves 32 particle slots with NQ + 1 warps (NQ = tabulated quantities: 4 Boozer, 7 cylindrical):
//   * the SCALAR warp: lane l owns particle slot l -- state, DP5 stage algebra, cell locate, the
//     guiding-centre physics, error norm, controller, stop test and refill.  Nothing is replicated:
//     one warp instruction advances 32 particles.
//   * NQ CONTRACTION warps: lane l of warp q owns the 64 tricubic coefficients of quantity q of slot l's
//     current cell, on chip (half in registers, half in a private conflict-free run of shared
//     memory), re-fetched from the cell-major table only when the slot's cell changes.  Per evaluation it
//     reads the slot's (cell, w) from shared memory, evaluates the 64-coefficient polynomial by nested
//     Horner (63 FMA, gc_device.cuh) and writes one value back.
// The two sides meet through named barriers (bar.arrive / bar.sync producer-consumer pairs): 1 = request
// published, 2 = values ready, 3 = guess published.  While the contraction warps work the scalar warp evaluates
// everything that does not need field values (the wave's exp / sincos, the next stage's partial sums, the
// known part of the error ratio) and GUESSES THE NEXT POINT'S CELL (fp32, straight-line extrapolation along
// the attempted step; at the end of an attempt from the accept/reject decision and the controller's new step
// length).  A contraction lane starts fetching the guessed cell as soon as it is done with the current point
// (eight 256-bit loads for the register half, one bulk asynchronous copy for the shared half), so the fetch
// overlaps the scalar warp's work; a wrong guess only costs a blocking fetch.  The seven stage derivatives,
// the step's start state and the per-particle bookkeeping live in shared memory, so the stage loop is rolled
// (one copy of the right-hand side in the instruction stream) and nothing spills.
#include <cstdlib>

#include "gc_device.cuh"

namespace catapult {

#ifndef CATAPULT_SPLIT_MINB_BOOZER
#define CATAPULT_SPLIT_MINB_BOOZER 4
#endif
#ifndef CATAPULT_SPLIT_MINB_CART
#define CATAPULT_SPLIT_MINB_CART 2
#endif

constexpr int MODE_ADAPTIVE = 0, MODE_SCRIPT = 1, MODE_STEP_ONCE = 2;

#ifdef CATAPULT_PF_STATS
__device__ unsigned long long g_blk[8];  // debugging aid: blocking fetches by request code
extern "C" int catapult_debug_blocking(unsigned long long* out8) {
  return cudaMemcpyFromSymbol(out8, g_blk, sizeof(g_blk)) != cudaSuccess;
}
#endif

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
  static constexpr int MINB = CART ? CATAPULT_SPLIT_MINB_CART : CATAPULT_SPLIT_MINB_BOOZER;
  // A contraction thread keeps the first 32 stored coefficients of its (cell, quantity) block (the rows j = 0, 1
  // of every slab, gc_device.cuh coef_row_pos) in registers and the other 32 in a private run of shared
  // memory: 256 bytes + 16 bytes of padding, so that the 8 lanes of a quarter warp reading 16 bytes each at
  // the same offset of their runs hit 8 different 16-byte bank groups.
  static constexpr int STRIP = 272;
  // shared-memory layout (bytes)
  static constexpr size_t OFF_COEF = 0;                              // [NCT] runs of STRIP bytes
  static constexpr size_t OFF_MBAR = OFF_COEF + (size_t)STRIP * NCT;  // uint64 [NCT]: one mbarrier per thread
  static constexpr size_t OFF_KS = OFF_MBAR + 8 * NCT;               // double [7][4][32]
  static constexpr size_t OFF_W = OFF_KS + 7 * 4 * 32 * 8;           // double [3][32]
  static constexpr size_t OFF_FV = OFF_W + 3 * 32 * 8;               // double [NQ][32]
  static constexpr size_t OFF_REQ = OFF_FV + (size_t)NQ * 32 * 8;    // int2   [32]: code, flat cell index
  static constexpr size_t OFF_POS = OFF_REQ + 32 * 8;                // float  [2][3][32]: last point, start point (cell units)
  static constexpr size_t OFF_GUESS = OFF_POS + 2 * 3 * 32 * 4;      // int    [2][32]: guessed cell of the next point, by round parity
  static constexpr size_t OFF_ERR = OFF_GUESS + 2 * 32 * 4;               // double [12][32]: known part of the error ratio; wave terms
  static constexpr size_t OFF_Y = OFF_ERR + 12 * 32 * 8;               // double [9][32]: state y at the start of the step, dt, stage partial sums
  static constexpr size_t OFF_COLD = OFF_Y + 9 * 32 * 8;                   // per-lane bookkeeping: 5 x int64[32] + 8 x int32[32]
  static constexpr size_t SMEM_BYTES = OFF_COLD + 5 * 256 + 8 * 128;
};

// Request of a slot: one word (what to evaluate: a stage point 0..5 of an attempted step, a start point, or
// nothing; whether the kernel ends) + the flat cell index, and the local coordinates w[3].  The guess of the
// NEXT point's cell travels separately (OFF_GUESS, barrier 3).
constexpr int REQ_NONE = -1, REQ_START = 6;
constexpr int CTL_PLAIN = 0, CTL_QUIT = 2;

__device__ __forceinline__ void bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ---- bulk asynchronous copy global -> shared (the TMA unit's 1-D form) with a thread-private mbarrier -------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned mbar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// this thread's arrival + the number of bytes the copy issued next will deliver
__device__ __forceinline__ void mbar_expect_tx(unsigned mbar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* gsrc, unsigned bytes, unsigned mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(gsrc), "r"(bytes), "r"(mbar)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned mbar, unsigned parity) {
  unsigned done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(mbar), "r"(parity)
        : "memory");
  } while (!done);
}

// the 64 bytes of one slab's two shared rows (j = 2: v[0..3], j = 3: v[4..7]) as one batch of loads
__device__ __forceinline__ void lds_slab(unsigned addr, double (&v)[8]) {
  asm volatile(
      "ld.shared.v2.f64 {%0,%1}, [%8];\n\t"
      "ld.shared.v2.f64 {%2,%3}, [%8+16];\n\t"
      "ld.shared.v2.f64 {%4,%5}, [%8+32];\n\t"
      "ld.shared.v2.f64 {%6,%7}, [%8+48];"
      : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3]), "=d"(v[4]), "=d"(v[5]), "=d"(v[6]), "=d"(v[7])
      : "r"(addr)
      : "memory");
}

// ---- contraction warps -----------------------------------------------------------------------------
// Where along the attempted step the next evaluation point lies, relative to this one, in units of
// (this point - start of the attempt): (c_next - c_this)/c_this for c = 1/5, 3/10, 4/5, 8/9, 1.
__constant__ float NEXT_POINT_RATIO[8] = {0.5f, 5.0f / 3.0f, 1.0f / 9.0f, 0.125f, 0.0f, 0.0f, 0.0f, 0.0f};
__device__ __forceinline__ float next_point_ratio(int r) { return NEXT_POINT_RATIO[r & 7]; }

// cell of the point pos + ratio (pos - base), all in cell units (fp32: this is only a guess).  Periodic
// dimensions: both points lie in [0, k), so the short way round differs from the plain difference by at most k.
template <int MODEL>
__device__ __forceinline__ int guess_cell(const FieldConst& f, const float pos[3], const float base[3], float ratio) {
  int ni[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const bool periodic = (d == 2) || (d == 1 && MODEL != MODEL_CART);
    const float kf = (float)f.k[d];
    float dd = pos[d] - base[d];
    if (periodic) dd = dd > 0.5f * kf ? dd - kf : (dd < -0.5f * kf ? dd + kf : dd);
    float p = fmaf(ratio, dd, pos[d]);
    if (periodic) p = p >= kf ? p - kf : (p < 0.f ? p + kf : p);
    ni[d] = min(max(__float2int_rd(p), 0), f.k[d] - 1);
  }
  return flat_cell(f, ni[0], ni[1], ni[2]);
}

template <int MODEL>
__device__ __forceinline__ void contraction_warp(const FieldConst& f, unsigned char* smem, int q, int lane,
                                                 unsigned long long* counters) {
  using ST = SplitTraits<MODEL>;
  constexpr int NQ = ST::NQ, NT = ST::NT;
  const double* __restrict__ table = f.table;
  double reg[32];
  unsigned char* strip = smem + ST::OFF_COEF + (size_t)(q * 32 + lane) * ST::STRIP;
  const unsigned strip_s = smem_u32(strip);
  const unsigned mbar = smem_u32(smem + ST::OFF_MBAR) + 8u * (q * 32 + lane);
  const double* wbuf = reinterpret_cast<const double*>(smem + ST::OFF_W);
  double* fvbuf = reinterpret_cast<double*>(smem + ST::OFF_FV);
  const volatile int2* reqbuf = reinterpret_cast<const volatile int2*>(smem + ST::OFF_REQ);
  const volatile int* guessbuf = reinterpret_cast<const volatile int*>(smem + ST::OFF_GUESS);
  int cached = -1;
  unsigned phase = 0;    // parity of the mbarrier phase the next wait is for
  bool pending = false;  // a bulk copy into the strip is in flight
#ifdef CATAPULT_PF_STATS
  unsigned long long n_block = 0, n_pref = 0;
#endif
  mbar_init(mbar, 1);

  // a cell's 512 contiguous bytes of this lane's quantity: the second half goes global -> shared as ONE bulk
  // asynchronous copy (no register staging, no per-16-byte requests), the first half lands in its final
  // registers.  Nothing waits here.
  auto wait_strip = [&]() {
    if (pending) {
      mbar_wait(mbar, phase);
      phase ^= 1u;
      pending = false;
    }
  };
  auto issue_loads = [&](int c) {
    const double* src = table + ((long long)c * NQ + q) * 64;
    // the eight vector loads first (they are the slower half: one request per 32 bytes), then the bulk copy
#pragma unroll
    for (int e = 0; e < 32; e += 4) ldg_f64x4(src + e, reg[e], reg[e + 1], reg[e + 2], reg[e + 3]);
    wait_strip();  // a wrong guess may still be landing in the strip: let it finish first
    mbar_expect_tx(mbar, 256);
    bulk_g2s(strip_s, src + 32, 256, mbar);
    pending = true;
  };
  for (;;) {
    bar_sync(1, NT);
    const long long rq_raw = *reinterpret_cast<const volatile long long*>(reqbuf + lane);  // one 8-byte load
    const int2 rq = make_int2((int)rq_raw, (int)(rq_raw >> 32));
    const int ctl = (rq.x >> 3) & 7;                            // block-uniform
    if (ctl == CTL_QUIT) break;
    const int code = (rq.x & 7) == 7 ? REQ_NONE : (rq.x & 7);
    // the local coordinates are loaded with the request, not after it has been looked at (one latency, not two)
    const double w0 = wbuf[lane], w1 = wbuf[32 + lane], w2 = wbuf[64 + lane];
    if (code >= 0) {
      const int c = rq.y;
      if (c != cached) {  // the guess missed (or there was none): one memory latency, paid by the whole block
        issue_loads(c);
        cached = c;
#ifdef CATAPULT_PF_STATS
        ++n_block;
        if (q == 0) atomicAdd(&g_blk[code & 7], 1ULL);
#endif
      }
      wait_strip();
      // horner64 (gc_device.cuh), same operations in the same order, scheduled by hand: the register half U
      // (8 independent rows) is worked while the first batch of the shared half is in flight; the shared
      // half V comes slab by slab, each slab's two rows as ONE batch of four 16-byte loads issued as soon as
      // the previous batch has been consumed
      double v[8];
      lds_slab(strip_s + 64 * 3, v);
      double U;
      {
        double pr[4];
#pragma unroll
        for (int g = 0; g < 2; ++g) {  // slabs 3,2 then 1,0: four rows at a time, level by level
          double a4[4];
#pragma unroll
          for (int r = 0; r < 4; ++r) a4[r] = fma(reg[(4 * (1 - g) + r) * 4 + 3], w2, reg[(4 * (1 - g) + r) * 4 + 2]);
#pragma unroll
          for (int r = 0; r < 4; ++r) a4[r] = fma(a4[r], w2, reg[(4 * (1 - g) + r) * 4 + 1]);
#pragma unroll
          for (int r = 0; r < 4; ++r) a4[r] = fma(a4[r], w2, reg[(4 * (1 - g) + r) * 4]);
          pr[2 * (1 - g) + 1] = fma(a4[3], w1, a4[2]);  // stored row = i*2 + j
          pr[2 * (1 - g)] = fma(a4[1], w1, a4[0]);
        }
        U = fma(fma(fma(pr[3], w0, pr[2]), w0, pr[1]), w0, pr[0]);
      }
      double V = 0.0;
#pragma unroll
      for (int i = 3; i >= 0; --i) {
        const double row1 = fma(fma(fma(v[7], w2, v[6]), w2, v[5]), w2, v[4]);
        const double row0 = fma(fma(fma(v[3], w2, v[2]), w2, v[1]), w2, v[0]);
        if (i > 0) lds_slab(strip_s + 64 * (i - 1), v);
        const double pair = fma(row1, w1, row0);
        V = (i == 3) ? pair : fma(V, w0, pair);
      }
      const double total = fma(V, w1 * w1, U);
      fvbuf[q * 32 + lane] = total;
    }
    __syncwarp();
    bar_arrive(2, NT);
    // ---- while the scalar warp works: it publishes its guess of the NEXT point's cell (barrier 3: in its
    // overlap window inside an attempted step; right after the accept/reject decision at its end); start
    // fetching that cell if it is not the one held.  A wrong guess costs what every cell change cost before
    // (a blocking fetch next round); a right one hides the fetch entirely.
    bar_sync(3, NT);
    int target = guessbuf[((rq.x >> 6) & 1) * 32 + lane];  // double-buffered by round parity
    if (code < 0 || target < 0) target = cached;
    if (target != cached) {
#ifdef CATAPULT_PF_STATS
      ++n_pref;
#endif
      issue_loads(target);
      cached = target;
    }
  }
#ifdef CATAPULT_PF_STATS
  if (counters && q == 0) {  // debugging aid: blocking / guessed fetches of quantity 0 in the two spare status counters
    atomicAdd(counters + 4, n_block);
    atomicAdd(counters + 5, n_pref);
  }
#else
  (void)counters;
#endif
}

// ---- scalar warp: geometry before the field values are known ------------------------------------------
struct EvalGeo {
  double a, inva, ang;                 // Boozer: s, 1/s, theta;  Cartesian: R, 1/R, phi
  double sn, cs, Phihat, dPhihat;      // wave terms (MODEL_BOOZER_SAW)
};

template <int MODEL>
__device__ __forceinline__ void eval_locate(const TraceConst& tc, const double y[4], int i[3], double w[3],
                                            float pos[3], EvalGeo& g) {
  const double r2 = fma(y[0], y[0], y[1] * y[1]);
  fm::sqrt_rsqrt(r2, g.a, g.inva);
  g.ang = fm::atan2(y[1], y[0]);
  if (MODEL == MODEL_CART) locate3<false>(tc.f, g.a, y[2], g.ang, i, w, pos);
  else locate3<true>(tc.f, g.a, g.ang, y[2], i, w, pos);
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

// sum_{j < NJ} a[NJ][j] k_j: the part of stage state NJ + 2 (row NJ of DP_A) that is known before k_NJ is
template <int NJ>
__device__ __forceinline__ void stage_partial(const double* ks, double* P) {  // P: shared, stride 32
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    double k[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) k[j] = ks[(j * 4 + c) * 32];  // the loads of a component first, then its sum
    double p = 0.0;
#pragma unroll
    for (int j = 0; j < NJ; ++j) p = fma(DP_A[NJ][j], k[j], p);
    P[c * 32] = p;
  }
}

// One lock-step evaluation round of the scalar warp, in two halves.  eval_publish: lanes with code >= 0 hand
// (cell indices, w) of the point (t, y) to the contraction warps; the others publish REQ_NONE.  eval_collect:
// picks up the interpolated values and finishes the right-hand side.  Between the two the caller may do
// anything that does not need field values (it overlaps the contraction).  All 32 lanes must call both.
template <int MODEL>
__device__ __forceinline__ void eval_publish(const TraceConst& tc, unsigned char* smem, int lane, int code, int ctl,
                                             int& rpar, double t, const double y[4], EvalGeo& g, float pos[3]) {
  using ST = SplitTraits<MODEL>;
  double* wbuf = reinterpret_cast<double*>(smem + ST::OFF_W);
  int2* reqbuf = reinterpret_cast<int2*>(smem + ST::OFF_REQ);
  float* posbuf = reinterpret_cast<float*>(smem + ST::OFF_POS);
  int i[3];
  double w[3];
  eval_locate<MODEL>(tc, y, i, w, pos, g);
  const int cell = flat_cell(tc.f, i[0], i[1], i[2]);
  wbuf[lane] = w[0];
  wbuf[32 + lane] = w[1];
  wbuf[64 + lane] = w[2];
  rpar ^= 1;  // round parity: selects the guess buffer of this round
  reqbuf[lane] = make_int2((code < 0 ? 7 : code) | (ctl << 3) | (rpar << 6), cell);  // one word: what to do + what follows
#pragma unroll
  for (int d = 0; d < 3; ++d) posbuf[d * 32 + lane] = pos[d];
  __syncwarp();
  bar_arrive(1, ST::NT);
  eval_wave<MODEL>(tc, t, y, g);
}

// the scalar warp's guess of the next evaluation point's cell (-1: none), handed over through barrier 3
template <int MODEL>
__device__ __forceinline__ void publish_guess(unsigned char* smem, int lane, int rpar, int target) {
  using ST = SplitTraits<MODEL>;
  reinterpret_cast<volatile int*>(smem + ST::OFF_GUESS)[rpar * 32 + lane] = target;
  __syncwarp();
  bar_arrive(3, ST::NT);
}

template <int MODEL>
__device__ __forceinline__ void eval_collect(const TraceConst& tc, unsigned char* smem, int lane, const double y[4],
                                             double mu, EvalGeo& g, double dy[4], double& modB, double& level) {
  using ST = SplitTraits<MODEL>;
  const double* fvbuf = reinterpret_cast<const double*>(smem + ST::OFF_FV);
  // The wave terms cross the barrier through shared memory: stores cannot move across a barrier, so the
  // arithmetic that produces them stays in the overlap window (ptxas otherwise sinks it below the barrier, onto
  // the critical path, to save the registers they would occupy across it).
  double* wavebuf = reinterpret_cast<double*>(smem + ST::OFF_ERR) + 8 * 32 + lane;
  if (MODEL == MODEL_BOOZER_SAW) {
    wavebuf[0] = g.sn;
    wavebuf[32] = g.cs;
    wavebuf[64] = g.Phihat;
    wavebuf[96] = g.dPhihat;
  }
  bar_sync(2, ST::NT);
  double fv[ST::NQ];
#pragma unroll
  for (int q = 0; q < ST::NQ; ++q) fv[q] = fvbuf[q * 32 + lane];
  if (MODEL == MODEL_BOOZER_SAW) {
    g.sn = wavebuf[0];
    g.cs = wavebuf[32];
    g.Phihat = wavebuf[64];
    g.dPhihat = wavebuf[96];
  }
  eval_physics<MODEL>(tc, y, mu, g, fv, dy, modB, level);
}

template <int MODEL>
__device__ __forceinline__ void eval_round(const TraceConst& tc, unsigned char* smem, int lane, int code, int& rpar,
                                           double t, const double y[4], double mu, double dy[4], double& modB,
                                           double& level) {
  using ST = SplitTraits<MODEL>;
  EvalGeo g;
  float pos[3];
  eval_publish<MODEL>(tc, smem, lane, code, CTL_PLAIN, rpar, t, y, g, pos);
  if (code >= 0) {  // a start point: the next attempted step is extrapolated from here
    float* basebuf = reinterpret_cast<float*>(smem + ST::OFF_POS) + 96;
#pragma unroll
    for (int d = 0; d < 3; ++d) basebuf[d * 32 + lane] = pos[d];
  }
  publish_guess<MODEL>(smem, lane, rpar, -1);
  eval_collect<MODEL>(tc, smem, lane, y, mu, g, dy, modB, level);
}

template <int MODEL, int MODE>
__global__ void __launch_bounds__(SplitTraits<MODEL>::NT, SplitTraits<MODEL>::MINB)
trace_kernel(const __grid_constant__ TraceConst tc, const __grid_constant__ TraceArgs a) {
  using ST = SplitTraits<MODEL>;
  extern __shared__ __align__(16) unsigned char smem[];
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  if (warp < ST::NQ) {
    contraction_warp<MODEL>(tc.f, smem, warp, lane, a.counters);
    return;
  }

  // ---- scalar warp ------------------------------------------------------------------------------------
  const unsigned FULL = 0xffffffffu;
  const long long n = a.n;
  double* ks = reinterpret_cast<double*>(smem + ST::OFF_KS) + lane;  // k_j component c at ks[(j*4+c)*32]
  double t = 0.0, mu = 0.0;
  double* ysm = reinterpret_cast<double*>(smem + ST::OFF_Y) + lane;  // y_c of the step's start at ysm[c * 32]
  double& dt = ysm[4 * 32];
  dt = 0.0;
  // bookkeeping that is touched once per attempted step or once per particle lives in shared memory, not in
  // registers (the compiler would spill it to local memory, whose reloads sat on the critical path)
  long long* cold64 = reinterpret_cast<long long*>(smem + ST::OFF_COLD) + lane;
  unsigned* cold32 = reinterpret_cast<unsigned*>(smem + ST::OFF_COLD + 5 * 256) + lane;
  long long& idx = cold64[0 * 32];
  long long& attempts_left = cold64[1 * 32];
  unsigned long long& c_acc = reinterpret_cast<unsigned long long&>(cold64[2 * 32]);
  unsigned long long& c_rej = reinterpret_cast<unsigned long long&>(cold64[3 * 32]);
  unsigned long long& c_eval = reinterpret_cast<unsigned long long&>(cold64[4 * 32]);
  unsigned& nacc = cold32[0 * 32];
  unsigned& nrej = cold32[1 * 32];
  int& consecutive = reinterpret_cast<int&>(cold32[2 * 32]);
  int& step = reinterpret_cast<int&>(cold32[3 * 32]);
  unsigned* c_fin = cold32 + 4 * 32;  // c_fin[s] at c_fin[s * 32]
  idx = -1;
  attempts_left = 0;
  c_acc = c_rej = c_eval = 0;
  nacc = nrej = 0;
  consecutive = step = 0;
#pragma unroll
  for (int j = 0; j < 4; ++j) c_fin[j * 32] = 0;
  bool active = false, exhausted = false;
  int rpar = 0;  // parity of the evaluation round (the guess buffer is double-buffered by it)

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
      eval_round<MODEL>(tc, smem, lane, fresh ? REQ_START : REQ_NONE, rpar, t, y, 0.0, dy0, B, level);
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
      // k1 with the particle's own mu: the field values are those of the round above; only the physics
      // is redone (mu enters linearly; the geometry is recomputed from y, cheap and rare)
      if (__any_sync(FULL, fresh && active)) {
        eval_round<MODEL>(tc, smem, lane, (fresh && active) ? REQ_START : REQ_NONE, rpar, t, y, mu, dy0, B, level);
        if (fresh && active) {
          ++c_eval;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            ks[c * 32] = dy0[c];
            ysm[c * 32] = y[c];
          }
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
      double* P = ysm + 5 * 32;  // sum_{j<st} a[st][j] k_j of the next stage, written in the overlap window
      double* errbuf = reinterpret_cast<double*>(smem + ST::OFF_ERR) + lane;  // [c]: sum, [4 + c]: 1/denominator
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        dy[c] = ks[c * 32];  // k1 (first-same-as-last, or the start point's derivative)
        P[c * 32] = 0.0;
      }
      EvalGeo g;
      // one stage point: its state, the request, and everything that overlaps the contraction
      auto stage_publish = [&](int st) {
        // stage state y + h sum_{j<=st} a[st][j] k_j (row 5 = b: the new state); the sum over j < st was
        // accumulated while the previous contraction ran, the newest derivative enters last
        const double ad = DP_A[st][st];
#pragma unroll
        for (int c = 0; c < 4; ++c) ys[c] = fma(h, fma(ad, dy[c], P[c * 32]), ysm[c * 32]);
        float pos[3];
        eval_publish<MODEL>(tc, smem, lane, stepping ? st : REQ_NONE, CTL_PLAIN, rpar, fma(DP_C[st], h, t), ys, g, pos);
        // ---- overlaps the contraction ----
        if (st < 5 || MODE == MODE_STEP_ONCE) {
          // the next point's cell, guessed by straight-line extrapolation from the step's start point (fp32,
          // cell units): the contraction warps start fetching it as soon as they are done with this point
          int target = -1;
          if (stepping && st < 5) {
            const float* basebuf = reinterpret_cast<const float*>(smem + ST::OFF_POS) + 96;
            const float base[3] = {basebuf[lane], basebuf[32 + lane], basebuf[64 + lane]};
            target = guess_cell<MODEL>(tc.f, pos, base, next_point_ratio(st));
          }
          publish_guess<MODEL>(smem, lane, rpar, target);
        }
        if (st < 5) {
          switch (st) {  // all the loads of a row first, then its sums (j ascending, as everywhere)
            case 0: stage_partial<1>(ks, P); break;
            case 1: stage_partial<2>(ks, P); break;
            case 2: stage_partial<3>(ks, P); break;
            case 3: stage_partial<4>(ks, P); break;
            default: stage_partial<5>(ks, P); break;
          }
        } else {
          // PAPER.md:85 Eq. 4, c = (1,1,1,v_total), state and derivative at the start of the
          // step: everything of the error ratio that does not need the last derivative
          const double ah = fabs(h);
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            double e = 0.0;
#pragma unroll
            for (int j = 0; j < 6; ++j)
              if (j != 1) e = fma(DP_E[j], ks[(j * 4 + c) * 32], e);
            errbuf[c * 32] = e;
            const double sc = (c == 3) ? tc.atol * tc.vtot : tc.atol;
            errbuf[(4 + c) * 32] = fm::rcp(fma(tc.rtol, fma(ah, fabs(ks[c * 32]), fabs(ysm[c * 32])), sc));
          }
        }
      };
      // The loop is cut between the overlap window and the pick-up of the values, so that the critical part of a
      // round (values -> physics -> next stage state -> locate -> request) is one straight-line block in which
      // the compiler can interleave the short critical chain with the rest.
      stage_publish(0);
#pragma unroll 1
      for (int st = 0; st < 5; ++st) {
        eval_collect<MODEL>(tc, smem, lane, ys, mu, g, dy, B_, level);
#pragma unroll
        for (int c = 0; c < 4; ++c) ks[((st + 1) * 4 + c) * 32] = dy[c];
        stage_publish(st + 1);
      }
      eval_collect<MODEL>(tc, smem, lane, ys, mu, g, dy, B_, level);
#pragma unroll
      for (int c = 0; c < 4; ++c) ks[(6 * 4 + c) * 32] = dy[c];
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
      else if (MODE == MODE_ADAPTIVE) dtn = controller(h, r, tc.dtmax, accepted);
      if (MODE != MODE_STEP_ONCE) {
        // the decision goes to the contraction warps at once, with the length of the next attempt over this
        // one's: they guess the cell of its first point (a rejected step is retried from the start point)
        double hn = h;
        if (MODE == MODE_ADAPTIVE) {
          const double tn = accepted ? (clamped ? tc.T : t + h) : t;
          hn = fmin((accepted && clamped) ? dt : dtn, tc.T - tn);
        }
        // first point of the next attempt: end point + ratio (end - start); accepted: a fifth of the next
        // step over this one beyond the end point, which becomes the new start point; rejected: the same,
        // measured from the start point
        const float fr = 0.2f * __fdividef((float)hn, (float)h);
        int target = -1;
        if (stepping) {
          float* posbuf = reinterpret_cast<float*>(smem + ST::OFF_POS);
          const float pe[3] = {posbuf[lane], posbuf[32 + lane], posbuf[64 + lane]};
          const float base[3] = {posbuf[96 + lane], posbuf[128 + lane], posbuf[160 + lane]};
          target = guess_cell<MODEL>(tc.f, pe, base, accepted ? fr : fr - 1.0f);
          if (accepted) {
#pragma unroll
            for (int d = 0; d < 3; ++d) posbuf[96 + d * 32 + lane] = pe[d];
          }
        }
        publish_guess<MODEL>(smem, lane, rpar, target);
      }
      if (stepping) {
        c_eval += 6;
        if (attempts_left > 0) --attempts_left;
        if (MODE == MODE_SCRIPT) {
          if (a.script_r) a.script_r[(long long)step * n + idx] = r;
          ++step;
        } else if (MODE == MODE_STEP_ONCE) {
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
              ysm[c * 32] = ys[c];
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
      ++c_fin[finish * 32];
      active = false;
    }
  }

  // release the contraction warps
  {
    reinterpret_cast<int2*>(smem + ST::OFF_REQ)[lane] = make_int2(7 | (CTL_QUIT << 3), 0);
    __syncwarp();
    bar_arrive(1, ST::NT);
  }

  // ---- statistics: one atomic per warp per counter -----------------------------------------------------
  if (a.counters) {
    unsigned long long v[7] = {c_acc, c_rej, c_fin[0], c_fin[32], c_fin[64], c_fin[96], c_eval};
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
  if (const char* e = getenv("CATAPULT_BLOCKS_PER_SM")) {  // experiments only
    const int v = atoi(e);
    if (v >= 1 && v < per_sm) per_sm = v;
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
