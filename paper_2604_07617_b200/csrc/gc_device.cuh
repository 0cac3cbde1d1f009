// Device-side arithmetic of the hot path: cell locate, local tricubic evaluation, the three
// guiding-centre right-hand sides and one Dormand-Prince 5(4) attempt.  fp64 throughout.
// Everything is __forceinline__ so that the DP5 stages stay in registers.
#pragma once

#include "internal.h"

namespace catapult {

constexpr int MODEL_BOOZER_VAC = 0;  // DESIGN.md R1
constexpr int MODEL_BOOZER_SAW = 1;  // DESIGN.md R2
constexpr int MODEL_CART = 2;        // DESIGN.md R3

template <int MODEL>
struct ModelTraits {
  static constexpr int NQ = (MODEL == MODEL_CART) ? CATAPULT_NQUANT_CYL : CATAPULT_NQUANT_BOOZER;
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

// reduces x-lo into [0, span) (periodic dimension)
__device__ __forceinline__ double wrap_periodic(double xr, double span, double invspan) {
  double r = fma(-span, floor(xr * invspan), xr);
  if (r < 0.0) r += span;
  if (r >= span) r -= span;
  if (!(r >= 0.0 && r < span)) r = 0.0;
  return r;
}

__device__ __forceinline__ int cell_and_u(double xr, double invh, int k, double& u) {
  const double t = xr * invh;
  double fi = floor(t);
  fi = fmin(fmax(fi, 0.0), (double)(k - 1));
  u = t - fi;
  return (int)fi;
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

__device__ __forceinline__ double2 ldg_f64x2(const double* p) {
  return __ldg(reinterpret_cast<const double2*>(p));
}

// ---- local tricubic evaluation of NQ quantities from one cell's [NQ][64] block ---------------
// sum_abc L0[a] L1[b] L2[c] F[a][b][c], contracted fastest index first (64 + 16 + 4 FMA).
template <int NQ>
__device__ __forceinline__ void tricubic_cell(const double* __restrict__ cellp, const double u[3], double out[NQ]) {
  double L0[4], L1[4], L2[4];
  lagrange4(u[0], L0);
  lagrange4(u[1], L1);
  lagrange4(u[2], L2);
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    double acc = 0.0;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      double sa = 0.0;
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const double2 f01 = ldg_f64x2(cellp + q * 64 + a * 16 + b * 4);
        const double2 f23 = ldg_f64x2(cellp + q * 64 + a * 16 + b * 4 + 2);
        double r = f01.x * L2[0];
        r = fma(f01.y, L2[1], r);
        r = fma(f23.x, L2[2], r);
        r = fma(f23.y, L2[3], r);
        sa = fma(r, L1[b], sa);
      }
      acc = fma(sa, L0[a], acc);
    }
    out[q] = acc;
  }
}

// ---- right-hand sides in the stepped variables ------------------------------------------------
// Boozer: y = (s cos th, s sin th, zeta, vpar); Cartesian: y = (x,y,z,vpar).
// `modB` = tabulated |B| at the point, `level` = s (Boozer) or interpolated psi (Cartesian).
template <int MODEL>
__device__ __forceinline__ void rhs(const TraceConst& tc, double t, const double y[4], double mu, double dy[4],
                                    double& modB, double& level, double* fv_out = nullptr) {
  const FieldConst& f = tc.f;
  constexpr int NQ = ModelTraits<MODEL>::NQ;
  double fv[NQ], u[3];
  if (MODEL == MODEL_CART) {
    const double R2 = fma(y[0], y[0], y[1] * y[1]);
    const double R = sqrt(R2);
    const double phi = atan2(y[1], y[0]);
    const long long cell = locate<false>(f, R, y[2], phi, u);
    tricubic_cell<NQ>(f.table + cell * (NQ * 64), u, fv);
    const double invR = 1.0 / R;
    const double cph = y[0] * invR, sph = y[1] * invR;
    const double BR = fv[0], Bp = fv[1], BZ = fv[2], gR = fv[3], gp = fv[4], gZ = fv[5];
    const double Bx = BR * cph - Bp * sph, By = BR * sph + Bp * cph, Bz = BZ;
    const double gx = gR * cph - gp * sph, gy = gR * sph + gp * cph, gz = gZ;
    const double B2 = fma(BR, BR, fma(Bp, Bp, BZ * BZ));
    const double B = sqrt(B2);
    const double invB = 1.0 / B;
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
    const double s = sqrt(s2);
    const double theta = atan2(y[1], y[0]);
    const long long cell = locate<true>(f, s, theta, y[2], u);
    tricubic_cell<NQ>(f.table + cell * (NQ * 64), u, fv);
    const double B = fv[0], B_s = fv[1], B_th = fv[2], B_ze = fv[3];
    const double vpar = y[3];
    const double invB = 1.0 / B;
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
      const double Phihat = tc.saw_Phi0 * exp(-ds * ds * tc.saw_invw2);
      const double dPhihat = Phihat * (-2.0 * ds * tc.saw_invw2);
      const double eta = fma(mm, theta, fma(-nn, y[2], om * t));
      double sn, cs;
      sincos(eta, &sn, &cs);
      const double Phi = Phihat * sn;
      const double Phi_psi = dPhihat * sn * f.invpsi0;
      const double Phi_th = mm * Phihat * cs;
      const double Phi_ze = -nn * Phihat * cs;
      const double kpar = fma(iota, mm, -nn);
      const double inv_omG = f.invG / om;
      const double al_th = -kpar * Phi_th * inv_omG;
      const double al_t = -kpar * Phihat * cs * f.invG;
      const double al_psi = -fma(f.iota1 * mm, Phi, kpar * dPhihat * sn) * inv_omG * f.invpsi0;
      const double psidot = fma(-B_th, W, fma(al_th, B * vpar, -Phi_th));
      sdot = psidot * f.invpsi0;
      const double iag = fma(-al_psi, f.G, iota);  // iota - alpha_psi G
      thdot = fma(B_psi, W, fma(iag * f.invG, vpar * B, Phi_psi));
      const double t1 = tc.M * mu * fma(al_th * B_psi, f.G, fma(B_th, iag, B_ze));
      const double t2 = tc.q * fma(al_t, f.G, fma(al_th * f.G, Phi_psi, fma(iag, Phi_th, Phi_ze)));
      vdot = fma(-(B * f.invG / tc.M), t1 + t2, vpar * invB * fma(B_th, Phi_psi, -B_psi * Phi_th));
    }
    const double invs = (s > 0.0) ? 1.0 / s : 0.0;
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
// kall (optional): all seven stage derivatives [7][4].
template <int MODEL, bool KALL>
__device__ __forceinline__ void dp5_attempt(const TraceConst& tc, double t, const double y[4], const double k1[4],
                                            double h, double mu, double ynew[4], double k7[4], double err[4],
                                            double& level_new, double* kall) {
  double k2[4], k3[4], k4[4], k5[4], k6[4], ys[4], B_, lv_;
#pragma unroll
  for (int i = 0; i < 4; ++i) ys[i] = fma(h, dp::a21 * k1[i], y[i]);
  rhs<MODEL>(tc, fma(dp::c2, h, t), ys, mu, k2, B_, lv_);
#pragma unroll
  for (int i = 0; i < 4; ++i) ys[i] = fma(h, fma(dp::a32, k2[i], dp::a31 * k1[i]), y[i]);
  rhs<MODEL>(tc, fma(dp::c3, h, t), ys, mu, k3, B_, lv_);
#pragma unroll
  for (int i = 0; i < 4; ++i) ys[i] = fma(h, fma(dp::a43, k3[i], fma(dp::a42, k2[i], dp::a41 * k1[i])), y[i]);
  rhs<MODEL>(tc, fma(dp::c4, h, t), ys, mu, k4, B_, lv_);
#pragma unroll
  for (int i = 0; i < 4; ++i)
    ys[i] = fma(h, fma(dp::a54, k4[i], fma(dp::a53, k3[i], fma(dp::a52, k2[i], dp::a51 * k1[i]))), y[i]);
  rhs<MODEL>(tc, fma(dp::c5, h, t), ys, mu, k5, B_, lv_);
#pragma unroll
  for (int i = 0; i < 4; ++i)
    ys[i] = fma(
        h, fma(dp::a65, k5[i], fma(dp::a64, k4[i], fma(dp::a63, k3[i], fma(dp::a62, k2[i], dp::a61 * k1[i])))),
        y[i]);
  rhs<MODEL>(tc, t + h, ys, mu, k6, B_, lv_);
#pragma unroll
  for (int i = 0; i < 4; ++i)
    ynew[i] = fma(
        h, fma(dp::b6, k6[i], fma(dp::b5, k5[i], fma(dp::b4, k4[i], fma(dp::b3, k3[i], dp::b1 * k1[i])))), y[i]);
  rhs<MODEL>(tc, t + h, ynew, mu, k7, B_, level_new);
#pragma unroll
  for (int i = 0; i < 4; ++i)
    err[i] = h * fma(dp::e7, k7[i],
                     fma(dp::e6, k6[i], fma(dp::e5, k5[i], fma(dp::e4, k4[i], fma(dp::e3, k3[i], dp::e1 * k1[i])))));
  if (KALL) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      kall[0 * 4 + i] = k1[i];
      kall[1 * 4 + i] = k2[i];
      kall[2 * 4 + i] = k3[i];
      kall[3 * 4 + i] = k4[i];
      kall[4 * 4 + i] = k5[i];
      kall[5 * 4 + i] = k6[i];
      kall[6 * 4 + i] = k7[i];
    }
  }
}

// PAPER.md:85 Eq. 4 with c = (1,1,1,v_total); state and derivative at the start of
// the step.  A non-finite component yields NaN, which the controller treats as a rejection.
__device__ __forceinline__ double error_ratio(const TraceConst& tc, const double err[4], const double y[4],
                                              const double k1[4], double h) {
  const double ah = fabs(h);
  double r = 0.0, chk = 0.0;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const double sc = (i == 3) ? tc.atol * tc.vtot : tc.atol;
    const double den = fma(tc.rtol, fma(ah, fabs(k1[i]), fabs(y[i])), sc);
    const double v = fabs(err[i]) / den;
    chk += v;
    r = fmax(r, v);
  }
  return (chk == chk) ? r : chk;
}

// Boost odeint default step adjuster for dopri5: see oracle/DESIGN.md S2.
__device__ __forceinline__ double controller(double h, double r, double dtmax, bool& accepted) {
  double dt = h;
  if (!(r <= 1.0)) {
    accepted = false;
    double fac = 0.9 * pow(r, -1.0 / 3.0);
    if (!(fac >= 0.2)) fac = 0.2;
    dt = h * fac;
  } else {
    accepted = true;
    if (r < 0.5) {
      const double rr = fmax(r, 1.0 / 3125.0);
      dt = h * 0.9 * pow(rr, -0.2);
    }
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
