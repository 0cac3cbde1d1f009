// Device-side arithmetic of the hot path: cell locate, local tricubic evaluation, the three
// guiding-centre right-hand sides and one Dormand-Prince 5(4) attempt.  fp64 throughout.
//
// Execution model: a particle is owned by a GROUP of NL consecutive lanes of a
// warp (NL = 4 by default).  Lane j of the group owns
//   - the 64 tricubic coefficients of quantity slots q = p*NL + j (p < QPL) of the particle's current
//     cell, cached on chip: the first NREG of them in registers, the rest in a private, bank-conflict-
//     free strip of shared memory.  A cell's 2 KiB (Boozer) / 3.5 KiB (Cartesian) are fetched from the
//     global table once per cell visit, not once per evaluation;
//   - state components c = i*NL + j (i < CPL) of the DP5 stage vectors k1..k7.
// The cheap scalar work (locate, Lagrange basis, physics) is replicated in the NL lanes; the 64-term
// contractions and the stage algebra are split between them and exchanged with warp shuffles.
// Everything is __forceinline__ so that the stages and the cached coefficients stay in registers.
#pragma once

#include "internal.h"
#include "gc_math.cuh"

namespace catapult {

constexpr int MODEL_BOOZER_VAC = 0;  // DESIGN.md R1
constexpr int MODEL_BOOZER_SAW = 1;  // DESIGN.md R2
constexpr int MODEL_CART = 2;        // DESIGN.md R3

// tunables (overridable with -D for sweeps; the defaults are the measured optimum)
#ifndef CATAPULT_NL_BOOZER
#define CATAPULT_NL_BOOZER 4
#endif
#ifndef CATAPULT_NREG_BOOZER
#define CATAPULT_NREG_BOOZER 32
#endif
#ifndef CATAPULT_MINB_BOOZER
#define CATAPULT_MINB_BOOZER 3
#endif
#ifndef CATAPULT_NL_CART
#define CATAPULT_NL_CART 4
#endif
#ifndef CATAPULT_NREG_CART
#define CATAPULT_NREG_CART 32
#endif
#ifndef CATAPULT_MINB_CART
#define CATAPULT_MINB_CART 2
#endif

constexpr int TRACE_THREADS = 128;

template <int MODEL>
struct ModelTraits {
  static constexpr bool CART = (MODEL == MODEL_CART);
  static constexpr int NQ = CART ? CATAPULT_NQUANT_CYL : CATAPULT_NQUANT_BOOZER;
  static constexpr int NL = CART ? CATAPULT_NL_CART : CATAPULT_NL_BOOZER;      // lanes per particle
  static constexpr int QPL = (NQ + NL - 1) / NL;                               // quantity slots per lane
  static constexpr int CPL = 4 / NL;                                           // state components per lane
  static constexpr int NREG = CART ? CATAPULT_NREG_CART : CATAPULT_NREG_BOOZER;  // coefficients in registers
  static constexpr int NSH = 64 * QPL - NREG;                                  // coefficients in shared memory
  static constexpr int MINB = CART ? CATAPULT_MINB_CART : CATAPULT_MINB_BOOZER;
  static constexpr int NT = TRACE_THREADS;
  static constexpr size_t SMEM_BYTES = (size_t)NT * NSH * sizeof(double);
  static_assert(NL == 1 || NL == 2 || NL == 4, "group size must be 1, 2 or 4");
  static_assert(NREG % 4 == 0 && NREG >= 0 && NREG <= 64 * QPL, "NREG must be a multiple of 4");
};

// ---- Dormand-Prince 5(4) tableau (ref [10] PAPER.md:164) -----------------------
namespace dp {
constexpr double c2 = 1.0 / 5.0, c3 = 3.0 / 10.0, c4 = 4.0 / 5.0, c5 = 8.0 / 9.0;
constexpr double a21 = 1.0 / 5.0;
constexpr double a31 = 3.0 / 40.0, a32 = 9.0 / 40.0;
constexpr double a41 = 44.0 / 45.0, a42 = -56.0 / 15.0, a43 = 32.0 / 9.0;
constexpr double a51 = 19372.0 / 6561.0, a52 = -25360.0 / 2187.0, a53 = 64448.0 / 6561.0, a54 = -212.0 / 729.0;
constexpr double a61 = 9017.0 / 3168.0, a62 = -355.0 / 33.0, a63 = 46732.0 / 5247.0, a64 = 49.0 / 176.0,
                 a65 = -5103.0 / 18656.0;
constexpr double b1 = 35.0 / 384.0, b3 = 500.0 / 1113.0, b4 = 125.0 / 192.0, b5 = -2187.0 / 6784.0,
                 b6 = 11.0 / 84.0;
// b - bhat
constexpr double e1 = 71.0 / 57600.0, e3 = -71.0 / 16695.0, e4 = 71.0 / 1920.0, e5 = -17253.0 / 339200.0,
                 e6 = 22.0 / 525.0, e7 = -1.0 / 40.0;
}  // namespace dp

// ---- lane group -----------------------------------------------------------------------------------
template <int NL>
struct Group {
  int j;           // lane within the group
  int gbase;       // first lane of the group within the warp
  unsigned gmask;  // lanes of the group
  __device__ __forceinline__ Group() {
    const int lane = threadIdx.x & 31;
    j = lane & (NL - 1);
    gbase = lane & ~(NL - 1);
    gmask = ((NL == 32) ? 0xffffffffu : ((1u << NL) - 1u)) << gbase;
  }
  // value held by lane jj of the group
  __device__ __forceinline__ double from(double v, int jj) const {
    return (NL == 1) ? v : __shfl_sync(gmask, v, gbase + jj);
  }
  __device__ __forceinline__ double max(double v) const {
#pragma unroll
    for (int o = NL / 2; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(gmask, v, o));
    return v;
  }
  __device__ __forceinline__ double sum(double v) const {
#pragma unroll
    for (int o = NL / 2; o > 0; o >>= 1) v += __shfl_xor_sync(gmask, v, o);
    return v;
  }
};

// component c = i*NL + j of a replicated 4-vector -> this lane's slot i (selects, no local memory)
template <int NL>
__device__ __forceinline__ double pick(const double full[4], int i, int j) {
  double r = full[i * NL];
#pragma unroll
  for (int jj = 1; jj < NL; ++jj) r = (j == jj) ? full[i * NL + jj] : r;
  return r;
}

// all-gather of the group's components: full[i*NL + jj] = slot i of lane jj
template <int NL, int CPL>
__device__ __forceinline__ void gather4(const Group<NL>& g, const double mine[CPL], double full[4]) {
#pragma unroll
  for (int i = 0; i < CPL; ++i)
#pragma unroll
    for (int jj = 0; jj < NL; ++jj) full[i * NL + jj] = g.from(mine[i], jj);
}

// ---- cell locate (nearest cell, cubic extrapolated outside) ---------------------
// Cubic Lagrange polynomials on the in-cell nodes {0,1/3,2/3,1}.
__device__ __forceinline__ void lagrange4(double u, double L[4]) {
  const double t1 = u - 1.0 / 3.0, t2 = u - 2.0 / 3.0, t3 = u - 1.0;
  const double p01 = u * t1, p23 = t2 * t3;
  L[0] = -4.5 * t1 * p23;
  L[1] = 13.5 * u * p23;
  L[2] = -13.5 * p01 * t3;
  L[3] = 4.5 * p01 * t2;
}

// reduces x-lo into [0, span) (periodic dimension).  span * floor(.) is exact inside the fma, so the result
// carries one rounding; a result that lands a rounding outside [0, span) is handled by the cell clamp
// (u marginally outside [0,1] on a face, where the two cells agree: DESIGN.md Q8, Q9).
__device__ __forceinline__ double wrap_periodic(double xr, double span, double invspan) {
  return fma(-span, floor(xr * invspan), xr);
}

// cell index clamped to [0, k-1] and local coordinate u = t - cell (outside [0,1] => extrapolation).
// The floor is taken by the fp64 -> int32 conversion (saturating; NaN -> 0) and clamped in integers.
__device__ __forceinline__ int cell_and_u(double xr, double invh, int k, double& u) {
  const double t = xr * invh;
  int i = __double2int_rd(t);
  i = min(max(i, 0), k - 1);
  u = t - (double)i;
  return i;
}

// x = grid coordinates (dim 0 never periodic; dim 1 periodic for Boozer; dim 2 always periodic)
template <bool DIM1_PERIODIC>
__device__ __forceinline__ long long locate(const FieldConst& f, double x0, double x1, double x2, double u[3]) {
  const int i0 = cell_and_u(x0 - f.lo[0], f.invh[0], f.k[0], u[0]);
  double r1 = x1 - f.lo[1];
  if (DIM1_PERIODIC) r1 = wrap_periodic(r1, f.span[1], f.invspan[1]);
  const int i1 = cell_and_u(r1, f.invh[1], f.k[1], u[1]);
  const double r2 = wrap_periodic(x2 - f.lo[2], f.span[2], f.invspan[2]);
  const int i2 = cell_and_u(r2, f.invh[2], f.k[2], u[2]);
  return ((long long)i0 * f.k[1] + i1) * f.k[2] + i2;
}

// 256-bit read-only global load (sm_100: LDG.E.256)
__device__ __forceinline__ void ldg_f64x4(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}

// ---- on-chip cache of the current cell's coefficients ----------------------------------------------
// Per lane: QPL*64 coefficients, element e = p*64 + (a*4+b)*4+c.  e < NREG lives in registers, the
// rest in shared memory as double2 chunks interleaved over the block's threads (chunk-major), so a
// quarter-warp LDS.128 reads 128 contiguous bytes: conflict-free, and private to the lane (no
// synchronisation is ever needed).
template <int MODEL>
struct CellCache {
  using MT = ModelTraits<MODEL>;
  double reg[MT::NREG > 0 ? MT::NREG : 1];
  double2* sl;     // this lane's strip: chunk c at sl[c * NT]
  long long cell;  // cached cell or -1

  __device__ __forceinline__ void init(double2* smem_base) {
    sl = smem_base + threadIdx.x;
    cell = -1;
  }

  // fetch the lane's quantity slots of `c` from the cell-major table [cell][quantity][64]
  __device__ __forceinline__ void load(const double* __restrict__ table, long long c, int j) {
    constexpr int NQ = MT::NQ, NL = MT::NL, QPL = MT::QPL, NREG = MT::NREG, NT = MT::NT;
#pragma unroll
    for (int p = 0; p < QPL; ++p) {
      int q = p * NL + j;
      if (q > NQ - 1) q = NQ - 1;  // padding slot (Cartesian: 7 quantities on 8 slots): a harmless duplicate
      const double* src = table + (c * NQ + q) * 64;
#pragma unroll
      for (int r = 0; r < 16; ++r) {
        double v0, v1, v2, v3;
        ldg_f64x4(src + 4 * r, v0, v1, v2, v3);
        const int e = p * 64 + 4 * r;
        if (e < NREG) {
          reg[e] = v0;
          reg[e + 1] = v1;
          reg[e + 2] = v2;
          reg[e + 3] = v3;
        } else {
          sl[((e - NREG) / 2) * NT] = make_double2(v0, v1);
          sl[((e - NREG) / 2 + 1) * NT] = make_double2(v2, v3);
        }
      }
    }
    cell = c;
  }

  __device__ __forceinline__ void ensure(const double* __restrict__ table, long long c, int j) {
    if (c != cell) load(table, c, j);
  }

  // sum_abc L0[a] L1[b] L2[c] F[a][b][c] for every quantity slot of the lane, contracted fastest index
  // first (64 + 16 + 4 FMA per quantity).
  __device__ __forceinline__ void contract(const double L0[4], const double L1[4], const double L2[4],
                                           double out[MT::QPL]) const {
    constexpr int QPL = MT::QPL, NREG = MT::NREG, NT = MT::NT;
#pragma unroll
    for (int p = 0; p < QPL; ++p) {
      double acc = 0.0;
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        double sa = 0.0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          const int e = p * 64 + a * 16 + b * 4;
          double f0, f1, f2, f3;
          if (e < NREG) {
            f0 = reg[e];
            f1 = reg[e + 1];
            f2 = reg[e + 2];
            f3 = reg[e + 3];
          } else {
            const double2 v01 = sl[((e - NREG) / 2) * NT];
            const double2 v23 = sl[((e - NREG) / 2 + 1) * NT];
            f0 = v01.x;
            f1 = v01.y;
            f2 = v23.x;
            f3 = v23.y;
          }
          double r = f0 * L2[0];
          r = fma(f1, L2[1], r);
          r = fma(f2, L2[2], r);
          r = fma(f3, L2[3], r);
          sa = fma(r, L1[b], sa);
        }
        acc = fma(sa, L0[a], acc);
      }
      out[p] = acc;
    }
  }
};

// tricubic values of all NQ quantities at local coordinates u of cell `c`, replicated in the group
template <int MODEL>
__device__ __forceinline__ void tricubic_group(const FieldConst& f, const Group<ModelTraits<MODEL>::NL>& g,
                                               CellCache<MODEL>& cc, long long c, const double u[3],
                                               double fv[ModelTraits<MODEL>::NQ]) {
  using MT = ModelTraits<MODEL>;
  cc.ensure(f.table, c, g.j);
  double L0[4], L1[4], L2[4], part[MT::QPL];
  lagrange4(u[0], L0);
  lagrange4(u[1], L1);
  lagrange4(u[2], L2);
  cc.contract(L0, L1, L2, part);
#pragma unroll
  for (int p = 0; p < MT::QPL; ++p)
#pragma unroll
    for (int jj = 0; jj < MT::NL; ++jj)
      if (p * MT::NL + jj < MT::NQ) fv[p * MT::NL + jj] = g.from(part[p], jj);
}

// ---- right-hand sides in the stepped variables ------------------------------------------------
// Boozer: y = (s cos th, s sin th, zeta, vpar); Cartesian: y = (x,y,z,vpar).
// y and dy are full 4-vectors replicated in the group.  `modB` = tabulated |B| at the point,
// `level` = s (Boozer) or interpolated psi (Cartesian).
template <int MODEL>
__device__ __forceinline__ void rhs(const TraceConst& tc, const Group<ModelTraits<MODEL>::NL>& g, CellCache<MODEL>& cc,
                                    double t, const double y[4], double mu, double dy[4], double& modB,
                                    double& level, double* fv_out = nullptr) {
  const FieldConst& f = tc.f;
  constexpr int NQ = ModelTraits<MODEL>::NQ;
  double fv[NQ], u[3];
  if (MODEL == MODEL_CART) {
    const double R2 = fma(y[0], y[0], y[1] * y[1]);
    double R, invR;
    fm::sqrt_rsqrt(R2, R, invR);
    const double phi = fm::atan2(y[1], y[0]);
    const long long cell = locate<false>(f, R, y[2], phi, u);
    tricubic_group<MODEL>(f, g, cc, cell, u, fv);
    const double cph = y[0] * invR, sph = y[1] * invR;
    const double BR = fv[0], Bp = fv[1], BZ = fv[2], gR = fv[3], gp = fv[4], gZ = fv[5];
    const double Bx = BR * cph - Bp * sph, By = BR * sph + Bp * cph, Bz = BZ;
    const double gx = gR * cph - gp * sph, gy = gR * sph + gp * cph, gz = gZ;
    const double B2 = fma(BR, BR, fma(Bp, Bp, BZ * BZ));
    double B, invB;
    fm::sqrt_rsqrt(B2, B, invB);
    const double vpar = y[3];
    // (M/(q|B|^3)) (vperp^2/2 + vpar^2),  vperp^2 = 2 mu |B|
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
    const double s2 = fma(y[0], y[0], y[1] * y[1]);
    double s, invs;
    fm::sqrt_rsqrt(s2, s, invs);
    const double theta = fm::atan2(y[1], y[0]);
    const long long cell = locate<true>(f, s, theta, y[2], u);
    tricubic_group<MODEL>(f, g, cc, cell, u, fv);
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
      // Phi = Phihat(s) sin(m th - n ze + w t); alpha = -(iota m - n) Phi / (w G)  (E_par = 0)
      const double mm = (double)tc.saw_m, nn = (double)tc.saw_n, om = tc.saw_omega;
      const double ds = s - tc.saw_s0;
      const double Phihat = tc.saw_Phi0 * fm::exp(-ds * ds * tc.saw_invw2);
      const double dPhihat = Phihat * (-2.0 * ds * tc.saw_invw2);
      const double eta = fma(mm, theta, fma(-nn, y[2], om * t));
      double sn, cs;
      fm::sincos(eta, sn, cs);
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
  if (fv_out) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) fv_out[q] = fv[q];
  }
}

// ---- one attempted DP5 step --------------------------------------------------------------------
// ynew = y + h sum b_i k_i, k7 = f(t+h, ynew) (first-same-as-last), err = h sum (b_i - bhat_i) k_i.
// y, ynew: full vectors replicated in the group; k1m, k7m, errm: this lane's CPL components
// (component c = i*NL + j).  kall_m (optional): all seven stage derivatives of the lane's components.
template <int MODEL, bool KALL>
__device__ __forceinline__ void dp5_attempt(const TraceConst& tc, const Group<ModelTraits<MODEL>::NL>& g,
                                            CellCache<MODEL>& cc, double t, const double y[4],
                                            const double k1m[ModelTraits<MODEL>::CPL], double h, double mu,
                                            double ynew[4], double k7m[ModelTraits<MODEL>::CPL],
                                            double errm[ModelTraits<MODEL>::CPL], double& level_new,
                                            double* kall_m) {
  constexpr int NL = ModelTraits<MODEL>::NL, CPL = ModelTraits<MODEL>::CPL;
  double k2m[CPL], k3m[CPL], k4m[CPL], k5m[CPL], k6m[CPL], ym[CPL], ysm[CPL], ys[4], dy[4], B_, lv_;
#pragma unroll
  for (int i = 0; i < CPL; ++i) ym[i] = pick<NL>(y, i, g.j);

#pragma unroll
  for (int i = 0; i < CPL; ++i) ysm[i] = fma(h, dp::a21 * k1m[i], ym[i]);
  gather4<NL, CPL>(g, ysm, ys);
  rhs<MODEL>(tc, g, cc, fma(dp::c2, h, t), ys, mu, dy, B_, lv_);
#pragma unroll
  for (int i = 0; i < CPL; ++i) k2m[i] = pick<NL>(dy, i, g.j);

#pragma unroll
  for (int i = 0; i < CPL; ++i) ysm[i] = fma(h, fma(dp::a32, k2m[i], dp::a31 * k1m[i]), ym[i]);
  gather4<NL, CPL>(g, ysm, ys);
  rhs<MODEL>(tc, g, cc, fma(dp::c3, h, t), ys, mu, dy, B_, lv_);
#pragma unroll
  for (int i = 0; i < CPL; ++i) k3m[i] = pick<NL>(dy, i, g.j);

#pragma unroll
  for (int i = 0; i < CPL; ++i)
    ysm[i] = fma(h, fma(dp::a43, k3m[i], fma(dp::a42, k2m[i], dp::a41 * k1m[i])), ym[i]);
  gather4<NL, CPL>(g, ysm, ys);
  rhs<MODEL>(tc, g, cc, fma(dp::c4, h, t), ys, mu, dy, B_, lv_);
#pragma unroll
  for (int i = 0; i < CPL; ++i) k4m[i] = pick<NL>(dy, i, g.j);

#pragma unroll
  for (int i = 0; i < CPL; ++i)
    ysm[i] = fma(h, fma(dp::a54, k4m[i], fma(dp::a53, k3m[i], fma(dp::a52, k2m[i], dp::a51 * k1m[i]))), ym[i]);
  gather4<NL, CPL>(g, ysm, ys);
  rhs<MODEL>(tc, g, cc, fma(dp::c5, h, t), ys, mu, dy, B_, lv_);
#pragma unroll
  for (int i = 0; i < CPL; ++i) k5m[i] = pick<NL>(dy, i, g.j);

#pragma unroll
  for (int i = 0; i < CPL; ++i)
    ysm[i] = fma(h,
                 fma(dp::a65, k5m[i],
                     fma(dp::a64, k4m[i], fma(dp::a63, k3m[i], fma(dp::a62, k2m[i], dp::a61 * k1m[i])))),
                 ym[i]);
  gather4<NL, CPL>(g, ysm, ys);
  rhs<MODEL>(tc, g, cc, t + h, ys, mu, dy, B_, lv_);
#pragma unroll
  for (int i = 0; i < CPL; ++i) k6m[i] = pick<NL>(dy, i, g.j);

#pragma unroll
  for (int i = 0; i < CPL; ++i)
    ysm[i] = fma(h,
                 fma(dp::b6, k6m[i],
                     fma(dp::b5, k5m[i], fma(dp::b4, k4m[i], fma(dp::b3, k3m[i], dp::b1 * k1m[i])))),
                 ym[i]);
  gather4<NL, CPL>(g, ysm, ynew);
  rhs<MODEL>(tc, g, cc, t + h, ynew, mu, dy, B_, level_new);
#pragma unroll
  for (int i = 0; i < CPL; ++i) k7m[i] = pick<NL>(dy, i, g.j);

#pragma unroll
  for (int i = 0; i < CPL; ++i)
    errm[i] = h * fma(dp::e7, k7m[i],
                      fma(dp::e6, k6m[i],
                          fma(dp::e5, k5m[i], fma(dp::e4, k4m[i], fma(dp::e3, k3m[i], dp::e1 * k1m[i])))));
  if (KALL) {
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
      kall_m[0 * CPL + i] = k1m[i];
      kall_m[1 * CPL + i] = k2m[i];
      kall_m[2 * CPL + i] = k3m[i];
      kall_m[3 * CPL + i] = k4m[i];
      kall_m[4 * CPL + i] = k5m[i];
      kall_m[5 * CPL + i] = k6m[i];
      kall_m[6 * CPL + i] = k7m[i];
    }
  }
}

// PAPER.md:85 Eq. 4 with c = (1,1,1,v_total); state and derivative at the start of
// the step.  Every lane scores its own components, the group takes the maximum.  A non-finite
// component yields NaN, which the controller treats as a rejection.
template <int NL, int CPL>
__device__ __forceinline__ double error_ratio(const TraceConst& tc, const Group<NL>& g, const double errm[CPL],
                                              const double y[4], const double k1m[CPL], double h) {
  const double ah = fabs(h);
  double r = 0.0, chk = 0.0;
#pragma unroll
  for (int i = 0; i < CPL; ++i) {
    const bool is_v = (i * NL + g.j == 3);
    const double sc = is_v ? tc.atol * tc.vtot : tc.atol;
    const double den = fma(tc.rtol, fma(ah, fabs(k1m[i]), fabs(pick<NL>(y, i, g.j))), sc);
    const double v = fabs(errm[i]) * fm::rcp(den);
    chk += v;
    r = fmax(r, v);
  }
  r = g.max(r);
  chk = g.sum(chk);
  return (chk == chk) ? r : chk;
}

// Boost odeint default step adjuster for dopri5 (S2):
//   r > 1  : reject, dt <- dt max(0.9 r^(-1/3), 1/5);  r < 0.5: accept, dt <- dt 0.9 max(r, 5^-5)^(-1/5).
// Both powers are taken by fm::pow_neg_inv on one code path (relative error ~1e-15, far below the
// sensitivity of anything downstream) so that lanes that grow and lanes that shrink do not diverge.
__device__ __forceinline__ double controller(double h, double r, double dtmax, bool& accepted) {
  accepted = (r <= 1.0);
  double dt = h;
  if (!accepted || r < 0.5) {
    const double base = accepted ? fmax(r, 1.0 / 3125.0) : r;
    double fac = 0.9 * fm::pow_neg_inv(base, accepted);
    if (!accepted && !(fac >= 0.2)) fac = 0.2;
    dt = h * fac;
  }
  return fmin(dt, dtmax);
}

// API state <-> stepped variables
template <int MODEL>
__device__ __forceinline__ void state_to_y(const double x[4], double y[4]) {
  if (MODEL == MODEL_CART) {
    y[0] = x[0]; y[1] = x[1]; y[2] = x[2]; y[3] = x[3];
  } else {
    double sn, cs;
    sincos(x[1], &sn, &cs);
    y[0] = x[0] * cs; y[1] = x[0] * sn; y[2] = x[2]; y[3] = x[3];
  }
}
template <int MODEL>
__device__ __forceinline__ void y_to_state(const double y[4], double x[4]) {
  if (MODEL == MODEL_CART) {
    x[0] = y[0]; x[1] = y[1]; x[2] = y[2]; x[3] = y[3];
  } else {
    x[0] = sqrt(fma(y[0], y[0], y[1] * y[1]));
    x[1] = atan2(y[1], y[0]);
    x[2] = y[2];
    x[3] = y[3];
  }
}

template <int MODEL>
__device__ __forceinline__ bool is_lost(const TraceConst& tc, double level) {
  return (MODEL == MODEL_CART) ? (level >= tc.f.psi0) : (level >= 1.0);
}

}  // namespace catapult
