// Device-side pieces shared by the kernels of libcatapult.so: cell locate, the tricubic contraction in
// the table's basis, the step-size controller, state conversions and the loss test.  fp64 throughout.
//
// Table basis: the local tricubic of PAPER.md:47-53 is stored per cell and
// quantity as its 64 coefficients in the centred monomials of the three local coordinates, w_d = 2 u_d - 1
// in [-1,1], not as its 64 nodal values: the interpolant is the same polynomial, its evaluation is a
// nested Horner scheme of 63 FMA on the three local coordinates alone (no Lagrange basis to build:
// 84 FMA + ~40 flops).  field.cu converts nodal values to this basis in double-double arithmetic, so
// every stored coefficient is the exact one rounded once.
//
// The three grid dimensions play three ROLES in the tracer (tracer.cu), named after the order in which a
// stage point's coordinates become known to the scalar warp:
//   FIRST  : the coordinate that is a state variable itself      (Boozer zeta = dim 2; cylindrical Z = dim 1)
//   SECOND : the one that needs a square root                    (Boozer s = dim 0;    cylindrical R = dim 0)
//   LAST   : the one that needs an arctangent                    (Boozer theta = dim 1; cylindrical phi = dim 2)
// Stored element (a*4 + b)*4 + c is the coefficient of wLAST^a wSECOND^b wFIRST^c: a run of four along c is a
// "row", the contraction runs FIRST -> SECOND -> LAST.
#pragma once

#include "gc_math.cuh"
#include "internal.h"

namespace catapult {

constexpr int MODEL_BOOZER_VAC = 0;  // DESIGN.md R1
constexpr int MODEL_BOOZER_SAW = 1;  // DESIGN.md R2
constexpr int MODEL_CART = 2;        // DESIGN.md R3
constexpr int MODEL_BOOZER_NV = 3;   // DESIGN.md R1b: non-vacuum Boozer, G(s), I(s), iota(s) tabulated

// ---- cell locate (nearest cell, cubic extrapolated outside) ---------------------
// reduces x-lo into [0, span) (periodic dimension).  span * floor(.) is exact inside the fma, so the result
// carries one rounding; a result that lands a rounding outside [0, span) is handled by the cell clamp
// (u marginally outside [0,1] on a face, where the two cells agree: DESIGN.md Q8, Q9).
__device__ __forceinline__ double wrap_periodic(double xr, double span, double invspan) {
  return fma(-span, floor(xr * invspan), xr);
}

// cell index clamped to [0, k-1] and centred local coordinate w = 2 (t - cell) - 1 (|w| > 1 => extrapolation,
// PAPER.md:79).  The floor is taken by the fp64 -> int32 conversion (saturating; NaN -> 0), clamped in integers.
__device__ __forceinline__ int cell_and_w(double xr, double invh, int k, double& w, float& pos) {
  const double t = xr * invh;
  int i = __double2int_rd(t);
  i = min(max(i, 0), k - 1);
  w = fma(2.0, t - (double)i, -1.0);
  pos = (float)t;  // position in cell units, for the tracer's next-cell guess only
  return i;
}
__device__ __forceinline__ int cell_and_w(double xr, double invh, int k, double& w) {
  float pos;
  return cell_and_w(xr, invh, k, w, pos);
}

// x = grid coordinates (dim 0 never periodic; dim 1 periodic for Boozer; dim 2 always periodic): per-dimension
// cell indices i[3], centred local coordinates w[3], position in cell units pos[3] (fp32)
template <bool DIM1_PERIODIC>
__device__ __forceinline__ void locate3(const FieldConst& f, double x0, double x1, double x2, int i[3], double w[3],
                                        float pos[3]) {
  i[0] = cell_and_w(x0 - f.lo[0], f.invh[0], f.k[0], w[0], pos[0]);
  double r1 = x1 - f.lo[1];
  if (DIM1_PERIODIC) r1 = wrap_periodic(r1, f.span[1], f.invspan[1]);
  i[1] = cell_and_w(r1, f.invh[1], f.k[1], w[1], pos[1]);
  const double r2 = wrap_periodic(x2 - f.lo[2], f.span[2], f.invspan[2]);
  i[2] = cell_and_w(r2, f.invh[2], f.k[2], w[2], pos[2]);
}
__device__ __forceinline__ int flat_cell(const FieldConst& f, int i0, int i1, int i2) {
  return (i0 * f.k[1] + i1) * f.k[2] + i2;
}
template <bool DIM1_PERIODIC>
__device__ __forceinline__ int locate(const FieldConst& f, double x0, double x1, double x2, double w[3]) {
  int i[3];
  float pos[3];
  locate3<DIM1_PERIODIC>(f, x0, x1, x2, i, w, pos);
  return flat_cell(f, i[0], i[1], i[2]);
}

// Which grid dimension plays which role (see the top of this file).
template <bool BOOZER>
struct AxisRoles {
  static constexpr int FIRST = BOOZER ? 2 : 1, SECOND = 0, LAST = BOOZER ? 1 : 2;
};
// Storage position of the coefficient of w0^p0 w1^p1 w2^p2 (powers per GRID dimension) inside a (cell, quantity)
// block of 64.  The first 32 stored coefficients (LAST-power 0, 1: 256 bytes) are the half a tracer thread keeps
// in registers, the other 32 (LAST-power 2, 3) the half it keeps in shared memory, fetched by ONE bulk copy.
__host__ __device__ constexpr int coef_pos(bool boozer, int p0, int p1, int p2) {
  return boozer ? (p1 * 4 + p0) * 4 + p2 : (p2 * 4 + p0) * 4 + p1;
}

// 256-bit read-only global load (sm_100: LDG.E.256)
__device__ __forceinline__ void ldg_f64x4(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}

// sum_abc C[(a*4+b)*4+c] wL^a wS^b wF^c.  get4(e, f0..f3) delivers the stored coefficients e..e+3 (a row) from
// wherever they live (registers, shared memory, global).  Every row by Horner in wF (3 FMA), the four rows of
// one LAST-power a by Horner in wS (3 FMA) -> plane value P_a, the four planes by Horner in wL (3 FMA):
// 48 + 12 + 3 = 63 FMA.  The tracer's contraction warps compute P_0..P_3 (they need only wF and wS), its
// scalar warp the last three FMA (tracer.cu); every user of the table evaluates it in this one order.
__device__ __forceinline__ double horner_row(double f0, double f1, double f2, double f3, double w) {
  return fma(fma(fma(f3, w, f2), w, f1), w, f0);
}
template <class Get4>
__device__ __forceinline__ double horner_plane(Get4 get4, int a, double wS, double wF) {
  double row[4];
#pragma unroll
  for (int b = 0; b < 4; ++b) {
    double f0, f1, f2, f3;
    get4((a * 4 + b) * 4, f0, f1, f2, f3);
    row[b] = horner_row(f0, f1, f2, f3, wF);
  }
  return horner_row(row[0], row[1], row[2], row[3], wS);
}
template <class Get4>
__device__ __forceinline__ double horner64(Get4 get4, double wL, double wS, double wF) {
  double P[4];
#pragma unroll
  for (int a = 0; a < 4; ++a) P[a] = horner_plane(get4, a, wS, wF);
  return horner_row(P[0], P[1], P[2], P[3], wL);
}

// A profile tabulated on the unique s-nodes (R1b): value and derivative with respect to s of the cubic
// through the four nodes of the s-cell (the tables' own piecewise-cubic interpolation; end cells extrapolate).
// u in cell units, invh = cells per unit of s.
__device__ __forceinline__ void profile_weights(double u, double invh, double L[4], double dL[4]) {
  const double t0 = u, t1 = u - 1.0 / 3.0, t2 = u - 2.0 / 3.0, t3 = u - 1.0;
  L[0] = -4.5 * t1 * t2 * t3;
  L[1] = 13.5 * t0 * t2 * t3;
  L[2] = -13.5 * t0 * t1 * t3;
  L[3] = 4.5 * t0 * t1 * t2;
  dL[0] = -4.5 * invh * (t2 * t3 + t1 * t3 + t1 * t2);
  dL[1] = 13.5 * invh * (t2 * t3 + t0 * t3 + t0 * t2);
  dL[2] = -13.5 * invh * (t1 * t3 + t0 * t3 + t0 * t1);
  dL[3] = 4.5 * invh * (t1 * t2 + t0 * t2 + t0 * t1);
}
__device__ __forceinline__ void profile_eval(const double* __restrict__ nodes, int cell, const double L[4],
                                             const double dL[4], double& v, double& dv) {
  const double* F = nodes + 3 * cell;
  const double f0 = __ldg(F), f1 = __ldg(F + 1), f2 = __ldg(F + 2), f3 = __ldg(F + 3);
  v = fma(L[3], f3, fma(L[2], f2, fma(L[1], f1, L[0] * f0)));
  dv = fma(dL[3], f3, fma(dL[2], f2, fma(dL[1], f1, dL[0] * f0)));
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

// API state <-> stepped variables.  Boozer: y = (s cos th, s sin th, zeta, vpar).
// Once per particle per call: the CUDA math library's full-range sincos / atan2 are used here.
template <int MODEL>
__device__ __forceinline__ void state_to_y(const double x[4], double y[4]) {
  if (MODEL == MODEL_CART) {
    y[0] = x[0]; y[1] = x[1]; y[2] = x[2]; y[3] = x[3];
  } else {
    double sn, cs;
    ::sincos(x[1], &sn, &cs);
    y[0] = x[0] * cs; y[1] = x[0] * sn; y[2] = x[2]; y[3] = x[3];
  }
}
template <int MODEL>
__device__ __forceinline__ void y_to_state(const double y[4], double x[4]) {
  if (MODEL == MODEL_CART) {
    x[0] = y[0]; x[1] = y[1]; x[2] = y[2]; x[3] = y[3];
  } else {
    x[0] = ::sqrt(fma(y[0], y[0], y[1] * y[1]));
    x[1] = ::atan2(y[1], y[0]);
    x[2] = y[2];
    x[3] = y[3];
  }
}

// Loss time inside the step that crossed the boundary (include/catapult.h loss_time_mode 1; S5b; Boozer:
// s = sqrt(y0^2 + y1^2)).  y(theta) is the cubic Hermite interpolant through the step's end states (ya, yb) and end
// derivatives (ka, kb; kb is the step's seventh stage), theta in [0, 1].  48 bisections from [0, 1] on "s(theta) >= 1":
// returns the smallest theta observed beyond the boundary and leaves y(theta) in yb.  Once per lost particle.
__device__ __forceinline__ void hermite_state(const double ya[4], const double ka[4], const double yb[4],
                                              const double kb[4], double h, double th, double y[4]) {
  const double t2 = th * th, t3 = t2 * th;
  const double h00 = 2.0 * t3 - 3.0 * t2 + 1.0, h10 = t3 - 2.0 * t2 + th, h01 = -2.0 * t3 + 3.0 * t2, h11 = t3 - t2;
#pragma unroll
  for (int i = 0; i < 4; ++i) y[i] = h00 * ya[i] + h10 * h * ka[i] + h01 * yb[i] + h11 * h * kb[i];
}
__device__ __forceinline__ double loss_refine_boozer(const double ya[4], const double ka[4], double yb[4],
                                                     const double kb[4], double h) {
  double lo = 0.0, hi = 1.0, ym[4];
#pragma unroll 1
  for (int it = 0; it < 48; ++it) {
    const double mid = 0.5 * (lo + hi);
    hermite_state(ya, ka, yb, kb, h, mid, ym);
    if (::sqrt(fma(ym[0], ym[0], ym[1] * ym[1])) >= 1.0) hi = mid;
    else lo = mid;
  }
  hermite_state(ya, ka, yb, kb, h, hi, ym);
#pragma unroll
  for (int i = 0; i < 4; ++i) yb[i] = ym[i];
  return hi;
}

template <int MODEL>
__device__ __forceinline__ bool is_lost(const TraceConst& tc, double level) {
  return (MODEL == MODEL_CART) ? (level >= tc.f.psi0) : (level >= 1.0);
}

}  // namespace catapult
