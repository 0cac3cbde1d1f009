// Device-side fp64 elementary functions of the tracer's scalar path, written for the argument ranges
// the guiding-centre right-hand sides produce.  The CUDA math
// library's atan2 / sincos / exp / pow / sqrt / division cover every IEEE corner (huge arguments,
// denormals, signed zeros, correctly rounded results) at 60-150 SASS instructions each; the profile of
// the first tracer showed them to be half of the instruction stream.  These versions keep <= ~2 ulp on the
// ranges used and cost 10-40 instructions.  Accuracy is checked on the GPU against numpy
// (tests/test_gpu_parity.py::test_device_math_parity).
#pragma once

#include "gc_math_coeffs.h"

namespace catapult {
namespace fm {

__device__ __forceinline__ int lo32(double x) { return __double2loint(x); }

// 1/x for finite normal x != 0: MUFU.RCP64H seed (~2^-20) + two Newton steps.  ~1 ulp.
__device__ __forceinline__ double rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}

// 1/sqrt(x) for finite normal x > 0: MUFU.RSQ64H seed + one third-order and one second-order step.
__device__ __forceinline__ double rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y * y, 1.0);                 // 1 - x y^2
  y = fma(y * e, fma(0.375, e, 0.5), y);          // y (1 + e/2 + 3 e^2/8)
  e = fma(-x, y * y, 1.0);
  y = fma(y * e, 0.5, y);
  return y;
}

// s = sqrt(x) and inv = 1/sqrt(x) together (x > 0).  x == 0 gives s = 0, inv = 0 (the caller's reading of
// the axis: cos = 1, sin = 0, R1).
__device__ __forceinline__ void sqrt_rsqrt(double x, double& s, double& inv) {
  const bool pos = x > 0.0;
  const double y = rsqrt(pos ? x : 1.0);
  double r = x * y;
  r = fma(fma(-r, r, x), 0.5 * y, r);             // one Heron correction: <= 1 ulp
  s = pos ? r : 0.0;
  inv = pos ? y : 0.0;
}

// atan2(y, x) in (-pi, pi]; (0,0) -> 0.  One division: the octant reduction picks numerator and
// denominator first, z = (mn - mx)/(mn + mx) when mn/mx > tan(pi/8), so that |z| <= tan(pi/8).
__device__ __forceinline__ double atan2(double y, double x) {
  const double ax = fabs(x), ay = fabs(y);
  const bool swap = ay > ax;
  const double mx = swap ? ay : ax, mn = swap ? ax : ay;
  const bool big = mn > 0.41421356237309503 * mx;
  const double num = big ? mn - mx : mn;
  double den = big ? mn + mx : mx;
  den = (den > 0.0) ? den : 1.0;
  const double z = num * rcp(den);
  const double w = z * z;
  double p = mathc::ATAN[mathc::N_ATAN - 1];
#pragma unroll
  for (int i = mathc::N_ATAN - 2; i >= 1; --i) p = fma(p, w, mathc::ATAN[i]);
  double r = fma(z * w, p, z);                    // z + z^3 P(z^2)
  r = big ? r + 0.78539816339744831 : r;          // + pi/4
  r = swap ? 1.5707963267948966 - r : r;
  r = (x < 0.0) ? 3.1415926535897931 - r : r;
  return copysign(r, y);
}

// sin and cos of x for |x| < ~2^30 (two-constant Cody-Waite reduction by pi/2; the products are exact
// inside the fma, so the reduced argument is good to ~1 ulp + |k| 2^-106).
__device__ __forceinline__ void sincos(double x, double& sn, double& cs) {
  const double MAGIC = 6755399441055744.0;        // 1.5 * 2^52: rint through the adder
  const double t = fma(x, 0.63661977236758138, MAGIC);
  const int q = lo32(t);
  const double k = t - MAGIC;
  double r = fma(-k, 1.5707963267948966, x);
  r = fma(-k, 6.123233995736766e-17, r);
  const double w = r * r;
  double ps = mathc::SIN[mathc::N_SIN - 1], pc = mathc::COS[mathc::N_COS - 1];
#pragma unroll
  for (int i = mathc::N_SIN - 2; i >= 0; --i) ps = fma(ps, w, mathc::SIN[i]);
#pragma unroll
  for (int i = mathc::N_COS - 2; i >= 0; --i) pc = fma(pc, w, mathc::COS[i]);
  const double s0 = fma(r * w, ps, r);                  // r + r^3 S(w)
  const double c0 = fma(w * w, pc, fma(-0.5, w, 1.0));  // 1 - w/2 + w^2 C(w)
  const bool odd = q & 1;
  double s1 = odd ? c0 : s0, c1 = odd ? s0 : c0;
  sn = (q & 2) ? -s1 : s1;
  cs = ((q + 1) & 2) ? -c1 : c1;
}

// exp(x) for x in [-700, 700] (clamped below; larger x is the caller's problem)
__device__ __forceinline__ double exp(double x) {
  const double MAGIC = 6755399441055744.0;
  x = (x > -700.0) ? x : -700.0;
  const double t = fma(x, 1.4426950408889634, MAGIC);
  const int k = lo32(t);
  const double kd = t - MAGIC;
  double r = fma(-kd, 0.69314718055994529, x);
  r = fma(-kd, 2.3190468138462996e-17, r);
  double p = mathc::EXP[mathc::N_EXP - 1];
#pragma unroll
  for (int i = mathc::N_EXP - 2; i >= 0; --i) p = fma(p, r, mathc::EXP[i]);
  p = fma(r * r, p, r) + 1.0;                     // 1 + r + r^2 E(r)
  return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}

// x^(-1/5) (five) or x^(-1/3) (!five) for x > 0: fp32 seed (MUFU.LG2 / MUFU.EX2, ~1e-6) + two Newton
// steps on y = x^(-1/n): y <- y + y (1 - x y^n)/n.  x = inf, x > FLT_MAX or NaN give NaN (the controller
// maps it to its floor).
__device__ __forceinline__ double pow_neg_inv(double x, bool five) {
  const float xf = __double2float_rn(x);
  const float yf = exp2f(__log2f(xf) * (five ? -0.2f : -0.33333334f));
  double y = (double)yf;
  const double invn = five ? 0.2 : (1.0 / 3.0);
#pragma unroll
  for (int it = 0; it < 2; ++it) {
    const double y2 = y * y;
    const double m = five ? y2 * y2 : y2;
    const double e = fma(-x, m * y, 1.0);
    y = fma(y * e, invn, y);
  }
  return y;
}

}  // namespace fm
}  // namespace catapult
