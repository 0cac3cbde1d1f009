// Pieces shared by the two tracer kernels (tracer_pair.cu: warp pairs, Boozer models; tracer.cu: one scalar warp +
// one contraction warp per quantity, cylindrical model): the Dormand-Prince tableau, the asynchronous-copy helpers,
// the next-cell guess and the guiding-centre right-hand sides (R1-R3).
#pragma once

#include "gc_device.cuh"

namespace catapult {

constexpr int MODE_ADAPTIVE = 0, MODE_SCRIPT = 1, MODE_STEP_ONCE = 2;

// Dormand-Prince 5(4) tableau for the rolled stage loop (row i = coefficients of the state fed to stage
// i+2; the last row is b: the 7th stage is evaluated at the new state).  PAPER.md:61, ref [10].
static __constant__ double DP_A[6][6] = {
    {1.0 / 5.0, 0, 0, 0, 0, 0},
    {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
static __constant__ double DP_C[6] = {1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
static __constant__ double DP_E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0, -17253.0 / 339200.0,
                               22.0 / 525.0, -1.0 / 40.0};
// Where along the attempted step the next evaluation point lies, relative to this one, in units of
// (this point - start of the attempt): (c_next - c_this)/c_this for c = 1/5, 3/10, 4/5, 8/9, 1; after the last
// point (the new state) the first point of the next attempt is guessed a fifth of a step further on.
static __constant__ float NEXT_POINT_RATIO[6] = {0.5f, 5.0f / 3.0f, 1.0f / 9.0f, 0.125f, 0.0f, 0.2f};

// Request word of a slot: bit 0 = the slot takes part in this round, bits 1-3 = kind of round (0..5: stage
// point of an attempted step; 6: a start point), bit 4 = the kernel ends, bit 6 = parity of the round.
constexpr int KIND_START = 6;
constexpr int REQ_QUIT = 1 << 4;

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

// one row (32 contiguous bytes) of the shared half
__device__ __forceinline__ void lds_row(unsigned addr, double (&v)[4]) {
  asm volatile(
      "ld.shared.v2.f64 {%0,%1}, [%4];\n\t"
      "ld.shared.v2.f64 {%2,%3}, [%4+16];"
      : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3])
      : "r"(addr)
      : "memory");
}
__device__ __forceinline__ void sts_f64x2(unsigned addr, double a, double b) {
  asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(addr), "d"(a), "d"(b) : "memory");
}

// sum_{j < NJ} a[NJ][j] k_j: the part of stage state NJ + 2 (row NJ of DP_A) that is known before k_NJ is
template <int NJ>
__device__ __forceinline__ double stage_partial(const double* ks) {  // ks: this lane's component, stride 128
  double k[NJ];
#pragma unroll
  for (int j = 0; j < NJ; ++j) k[j] = ks[j * 128];  // the loads first, then the sum (j ascending, as everywhere)
  double p = 0.0;
#pragma unroll
  for (int j = 0; j < NJ; ++j) p = fma(DP_A[NJ][j], k[j], p);
  return p;
}

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

// (c + i s)^m for an integer m (block-uniform): cos and sin of m times the angle whose cosine and sine are c, s
__device__ __forceinline__ void unit_power(int m, double c, double s, double& cm, double& sm) {
  if (m == 1) {
    cm = c;
    sm = s;
    return;
  }
  double bc = c, bs = s;
  cm = 1.0;
  sm = 0.0;
  for (unsigned k = (unsigned)(m < 0 ? -m : m); k; k >>= 1) {
    if (k & 1u) {
      const double t = fma(cm, bc, -sm * bs);
      sm = fma(cm, bs, sm * bc);
      cm = t;
    }
    const double t = fma(bc, bc, -bs * bs);
    bs = 2.0 * bc * bs;
    bc = t;
  }
  if (m < 0) sm = -sm;
}

struct EvalGeo {
  double a, inva;                  // Boozer: s, 1/s;  Cartesian: R, 1/R
  double ca, sa;                   // cosine and sine of theta (phi): y0/a, y1/a
  double sn, cs, Phihat, dPhihat;  // wave terms (MODEL_BOOZER_SAW)
  // ... and what the right-hand side makes of them without the field values (eval_wave_terms)
  double Phi_psi, Phi_th, al_th, iag, iagG, t2;
  // non-vacuum Boozer (MODEL_BOOZER_NV): G, dG/dpsi, I, dI/dpsi, iota at s (eval_profiles)
  double Gs, Gp, Is, Ip, io;
};

// The profiles of R1b at s (R1b): needs only s, so it runs while the contraction does.
__device__ __forceinline__ void eval_profiles(const FieldConst& f, EvalGeo& g) {
  const double t = (g.a - f.lo[0]) * f.invh[0];
  int i = __double2int_rd(t);
  i = min(max(i, 0), f.k[0] - 1);
  double L[4], dL[4], dG, dI, dio;
  profile_weights(t - (double)i, f.invh[0], L, dL);
  const int np = 3 * f.k[0] + 1;
  profile_eval(f.prof, i, L, dL, g.Gs, dG);
  profile_eval(f.prof + np, i, L, dL, g.Is, dI);
  profile_eval(f.prof + 2 * np, i, L, dL, g.io, dio);
  g.Gp = dG * f.invpsi0;
  g.Ip = dI * f.invpsi0;
}

// The part of R2 that does not need the interpolated field: computed while the
// contraction is still running.  Same operations, same order as if written inside eval_physics.
__device__ __forceinline__ void eval_wave_terms(const TraceConst& tc, EvalGeo& g) {
  const FieldConst& f = tc.f;
  const double mm = (double)tc.saw_m, nn = (double)tc.saw_n;
  const double Phihat = g.Phihat, dPhihat = g.dPhihat, sn = g.sn, cs = g.cs;
  const double iota = fma(f.iota1, g.a, f.iota0);
  const double Phi = Phihat * sn;
  g.Phi_psi = dPhihat * sn * f.invpsi0;
  g.Phi_th = mm * Phihat * cs;
  const double Phi_ze = -nn * Phihat * cs;
  const double kpar = fma(iota, mm, -nn);
  const double inv_omG = tc.saw_inv_omG;
  g.al_th = -kpar * g.Phi_th * inv_omG;
  const double al_t = -kpar * Phihat * cs * f.invG;
  const double al_psi = -fma(f.iota1 * mm, Phi, kpar * dPhihat * sn) * inv_omG * f.invpsi0;
  g.iag = fma(-al_psi, f.G, iota);  // iota - alpha_psi G
  g.iagG = g.iag * f.invG;
  g.t2 = tc.q * fma(al_t, f.G, fma(g.al_th * f.G, g.Phi_psi, fma(g.iag, g.Phi_th, Phi_ze)));
}

// DESIGN.md R1-R3 with the interpolated values fv
template <int MODEL>
__device__ __forceinline__ void eval_physics(const TraceConst& tc, const double y[4], double mu, const EvalGeo& g,
                                             const double* fv, double dy[4], double& modB, double& level) {
  const FieldConst& f = tc.f;
  if (MODEL == MODEL_CART) {
    const double cph = g.ca, sph = g.sa;
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
    const double s = g.a;
    const double B = fv[0], B_s = fv[1], B_th = fv[2], B_ze = fv[3];
    const double vpar = y[3];
    const double invB = fm::rcp(B);
    const double W = tc.Moq * fma(vpar * vpar, invB, mu);
    const double iota = fma(f.iota1, s, f.iota0);
    const double B_psi = B_s * f.invpsi0;
    const double vBG = vpar * B * f.invG;
    double sdot, thdot, vdot;
    if (MODEL == MODEL_BOOZER_NV) {
      // R1b: D = G + iota I + rho (G I' - I G'), rho = M vpar / (q B), ' = d/dpsi
      const double rho = tc.Moq * vpar * invB;
      const double D = fma(rho, fma(g.Gs, g.Ip, -g.Is * g.Gp), fma(g.io, g.Is, g.Gs));
      const double invD = fm::rcp(D);
      const double ca = fma(-rho, g.Gp, g.io), cb = fma(rho, g.Ip, 1.0);
      const double vB = vpar * B;
      sdot = -W * fma(g.Gs, B_th, -g.Is * B_ze) * invD * f.invpsi0;
      thdot = fma(g.Gs * W, B_psi, ca * vB) * invD;
      const double zedot = fma(cb, vB, -g.Is * W * B_psi) * invD;
      vdot = -mu * B * fma(ca, B_th, cb * B_ze) * invD;
      dy[0] = fma(sdot, g.ca, -thdot * y[1]);
      dy[1] = fma(sdot, g.sa, thdot * y[0]);
      dy[2] = zedot;
      dy[3] = vdot;
      modB = B;
      level = s;
      return;
    }
    if (MODEL == MODEL_BOOZER_VAC) {
      sdot = -B_th * W * f.invpsi0;
      thdot = fma(B_psi, W, iota * vBG);
      vdot = -fma(iota, B_th, B_ze) * mu * B * f.invG;
    } else {
      // the wave's own terms come from eval_wave_terms (the caller has run it for this point)
      const double Phi_psi = g.Phi_psi, Phi_th = g.Phi_th, al_th = g.al_th, iag = g.iag;
      const double psidot = fma(-B_th, W, fma(al_th, B * vpar, -Phi_th));
      sdot = psidot * f.invpsi0;
      thdot = fma(B_psi, W, fma(g.iagG, vpar * B, Phi_psi));
      const double t1 = tc.M * mu * fma(al_th * B_psi, f.G, fma(B_th, iag, B_ze));
      vdot = fma(-(B * f.invG * tc.invM), t1 + g.t2, vpar * invB * fma(B_th, Phi_psi, -B_psi * Phi_th));
    }
    dy[0] = fma(sdot, g.ca, -thdot * y[1]);
    dy[1] = fma(sdot, g.sa, thdot * y[0]);
    dy[2] = vBG;
    dy[3] = vdot;
    modB = B;
    level = s;
  }
}

// tracer_pair.cu
catapult_status launch_trace_pair(const TraceConst& tc, const TraceArgs& a, int model, int mode, cudaStream_t s);
catapult_status trace_pair_shape(int model, bool doi, int64_t n, int* blocks, int* threads);

}  // namespace catapult
