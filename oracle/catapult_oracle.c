/*
 * CATAPULT oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see catapult_oracle.h).
 *
 * Plain scalar double precision, no blocking, no fusion, no reordering beyond what
 * PAPER.md / DESIGN.md state.  Compiled with -O2 -ffp-contract=off (no fast-math).
 */
#include "catapult_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846
#define ORC_E_CHARGE 1.602176634e-19

/* ------------------------------------------------------------------------------------------
 * Local tricubic interpolation ("4x4x4 grid of points covering the cell",
 * PAPER.md:69 "(3k+1)^3 unique nodes").  Cubic Lagrange polynomials on the in-cell nodes
 * {0, 1/3, 2/3, 1}.
 * ---------------------------------------------------------------------------------------- */
void orc_lagrange4(double u, double L[4]) {
  const double t0 = u, t1 = u - 1.0 / 3.0, t2 = u - 2.0 / 3.0, t3 = u - 1.0;
  L[0] = -(9.0 / 2.0) * t1 * t2 * t3;
  L[1] = (27.0 / 2.0) * t0 * t2 * t3;
  L[2] = -(27.0 / 2.0) * t0 * t1 * t3;
  L[3] = (9.0 / 2.0) * t0 * t1 * t2;
}

/* derivative of the cubic Lagrange basis on {0, 1/3, 2/3, 1} with respect to u */
void orc_dlagrange4(double u, double dL[4]) {
  const double t0 = u, t1 = u - 1.0 / 3.0, t2 = u - 2.0 / 3.0, t3 = u - 1.0;
  dL[0] = -(9.0 / 2.0) * (t2 * t3 + t1 * t3 + t1 * t2);
  dL[1] = (27.0 / 2.0) * (t2 * t3 + t0 * t3 + t0 * t2);
  dL[2] = -(27.0 / 2.0) * (t1 * t3 + t0 * t3 + t0 * t1);
  dL[3] = (9.0 / 2.0) * (t1 * t2 + t0 * t2 + t0 * t1);
}

/* A profile given on the unique s-nodes (iota "is represented on a regular interpolant grid"):
   the cell of s as in orc_locate (clamped: the end cells' cubics are extrapolated), value and
   derivative with respect to s of that cell's cubic through its four nodes. */
void orc_profile(const orc_field *f, const double *nodes, double s, double *val, double *dval_ds) {
  const int k = f->ncell[0];
  const double h = (f->hi[0] - f->lo[0]) / (double)k;
  const double t = (s - f->lo[0]) / h;
  double fi = floor(t);
  if (fi < 0.0) fi = 0.0;
  if (fi > (double)(k - 1)) fi = (double)(k - 1);
  const double u = t - fi;
  double L[4], dL[4];
  orc_lagrange4(u, L);
  orc_dlagrange4(u, dL);
  const double *F = nodes + 3 * (int64_t)fi;
  double v = 0.0, d = 0.0;
  for (int a = 0; a < 4; ++a) {
    v += L[a] * F[a];
    d += dL[a] * F[a];
  }
  *val = v;
  *dval_ds = d / h;
}

static int orc_is_periodic(const orc_field *f, int d) {
  if (f->coord == ORC_COORD_BOOZER) return d >= 1; /* theta, zeta */
  return d == 2;                                   /* phi */
}

/* outside the grid the nearest cell's data is used "as if the particle was inside
   the cell" => the clamp leaves u outside [0,1] and the cubic is extrapolated.
   Periodic dims are first reduced into [lo,hi) (reading Q9). */
void orc_locate(const orc_field *f, const double x[3], int32_t cell[3], double u[3]) {
  for (int d = 0; d < 3; ++d) {
    const int k = f->ncell[d];
    const double span = f->hi[d] - f->lo[d];
    const double h = span / (double)k;
    double xr = x[d] - f->lo[d];
    if (orc_is_periodic(f, d)) {
      xr = xr - span * floor(xr / span);
      if (xr >= span || xr < 0.0) xr = 0.0;
    }
    const double t = xr / h;
    double fi = floor(t);
    if (fi < 0.0) fi = 0.0;
    if (fi > (double)(k - 1)) fi = (double)(k - 1);
    cell[d] = (int32_t)fi;
    u[d] = t - fi;
  }
}

void orc_tricubic(const orc_field *f, const double x[3], double *out) {
  if (f->analytic) {
    f->analytic(f->analytic_ctx, x, out);
    return;
  }
  int32_t cell[3];
  double u[3], L0[4], L1[4], L2[4];
  orc_locate(f, x, cell, u);
  orc_lagrange4(u[0], L0);
  orc_lagrange4(u[1], L1);
  orc_lagrange4(u[2], L2);
  const int64_t n0 = 3 * (int64_t)f->ncell[0] + 1, n1 = 3 * (int64_t)f->ncell[1] + 1,
                n2 = 3 * (int64_t)f->ncell[2] + 1;
  for (int q = 0; q < f->nquant; ++q) {
    const double *F = f->nodes + (int64_t)q * n0 * n1 * n2;
    double acc = 0.0;
    for (int a = 0; a < 4; ++a)
      for (int b = 0; b < 4; ++b)
        for (int c = 0; c < 4; ++c) {
          const int64_t j0 = 3 * (int64_t)cell[0] + a, j1 = 3 * (int64_t)cell[1] + b,
                        j2 = 3 * (int64_t)cell[2] + c;
          acc += L0[a] * L1[b] * L2[c] * F[(j0 * n1 + j1) * n2 + j2];
        }
    out[q] = acc;
  }
}

/* DESIGN.md reading R1c: the gradient of the SAME local tricubic, obtained by differentiating the
   Lagrange basis along one axis at a time; d/dx_d = (d/du_d) / h_d. */
void orc_tricubic_grad(const orc_field *f, const double x[3], int q, double *val, double grad[3]) {
  int32_t cell[3];
  double u[3], L[3][4], dL[3][4];
  orc_locate(f, x, cell, u);
  for (int d = 0; d < 3; ++d) {
    orc_lagrange4(u[d], L[d]);
    orc_dlagrange4(u[d], dL[d]);
  }
  const int64_t n0 = 3 * (int64_t)f->ncell[0] + 1, n1 = 3 * (int64_t)f->ncell[1] + 1,
                n2 = 3 * (int64_t)f->ncell[2] + 1;
  const double *F = f->nodes + (int64_t)q * n0 * n1 * n2;
  double v = 0.0, g0 = 0.0, g1 = 0.0, g2 = 0.0;
  for (int a = 0; a < 4; ++a)
    for (int b = 0; b < 4; ++b)
      for (int c = 0; c < 4; ++c) {
        const int64_t j0 = 3 * (int64_t)cell[0] + a, j1 = 3 * (int64_t)cell[1] + b, j2 = 3 * (int64_t)cell[2] + c;
        const double Fv = F[(j0 * n1 + j1) * n2 + j2];
        v += L[0][a] * L[1][b] * L[2][c] * Fv;
        g0 += dL[0][a] * L[1][b] * L[2][c] * Fv;
        g1 += L[0][a] * dL[1][b] * L[2][c] * Fv;
        g2 += L[0][a] * L[1][b] * dL[2][c] * Fv;
      }
  *val = v;
  for (int d = 0; d < 3; ++d) {
    const double h = (f->hi[d] - f->lo[d]) / (double)f->ncell[d];
    grad[d] = (d == 0 ? g0 : (d == 1 ? g1 : g2)) / h;
  }
}

void orc_tricubic_many(const orc_field *f, int64_t npts, const double *pts, double *out) {
  for (int64_t i = 0; i < npts; ++i) {
    double x[3] = {pts[i], pts[npts + i], pts[2 * npts + i]};
    double v[16];
    orc_tricubic(f, x, v);
    for (int q = 0; q < f->nquant; ++q) out[(int64_t)q * npts + i] = v[q];
  }
}

/* rows = nodes, columns = quantities; the 64 rows of a cell contiguous; cells and
   in-cell nodes ordered dim0, dim1, dim2 slowest -> fastest; boundary nodes stored redundantly. */
void orc_field_build(const orc_field *f, double *out) {
  const int64_t n0 = 3 * (int64_t)f->ncell[0] + 1, n1 = 3 * (int64_t)f->ncell[1] + 1,
                n2 = 3 * (int64_t)f->ncell[2] + 1;
  const int m = f->nquant;
  int64_t row = 0;
  for (int i0 = 0; i0 < f->ncell[0]; ++i0)
    for (int i1 = 0; i1 < f->ncell[1]; ++i1)
      for (int i2 = 0; i2 < f->ncell[2]; ++i2)
        for (int a = 0; a < 4; ++a)
          for (int b = 0; b < 4; ++b)
            for (int c = 0; c < 4; ++c) {
              const int64_t j0 = 3 * i0 + a, j1 = 3 * i1 + b, j2 = 3 * i2 + c;
              for (int q = 0; q < m; ++q)
                out[row * m + q] = f->nodes[(int64_t)q * n0 * n1 * n2 + (j0 * n1 + j1) * n2 + j2];
              ++row;
            }
}

/* ------------------------------------------------------------------------------------------
 * Guiding-centre equations: Euler-Lagrange equations of the Littlejohn Lagrangian
 * (Eq. 3) in Boozer form A = psi grad(theta) - psi_p grad(zeta),
 * B = G grad(zeta) + I grad(theta), dpsi_p/dpsi = iota (R1, R2).
 * mu is the magnetic moment per unit mass, mu = vperp^2/(2B) (PAPER.md:41 with M factored out).
 * Vacuum: I = 0, G constant.
 * ---------------------------------------------------------------------------------------- */
void orc_gc_boozer(const orc_field *f, const orc_params *p, double mu, double t, double s,
                   double theta, double zeta, double vpar, const double fv[4], double out[4]) {
  const double M = p->mass, q = p->charge;
  const double B = fv[0], B_s = fv[1], B_th = fv[2], B_ze = fv[3];
  const double G = f->G0, psi0 = f->psi0;
  const double iota = f->iota0 + f->iota1 * s;
  const double W = (M / q) * (vpar * vpar / B + mu);
  const double B_psi = B_s / psi0;
  if (f->G_nodes) {
    /* R1b (non-vacuum Boozer, no wave): Euler-Lagrange equations of Eq. 3 with B = G(psi) grad(zeta) +
       I(psi) grad(theta), A = psi grad(theta) - psi_p grad(zeta), dpsi_p/dpsi = iota; ' = d/dpsi:
         D = G + iota I + rho (G I' - I G'),  rho = M vpar / (q B)
         psidot = -W (G B_th - I B_ze) / D
         thdot  = (G W B_psi + (iota - rho G') vpar B) / D
         zedot  = ((1 + rho I') vpar B - I W B_psi) / D
         vdot   = -mu B ((iota - rho G') B_th + (1 + rho I') B_ze) / D                                  */
    double Gs, dG, Is, dI, io, dio;
    orc_profile(f, f->G_nodes, s, &Gs, &dG);
    orc_profile(f, f->I_nodes, s, &Is, &dI);
    orc_profile(f, f->iota_nodes, s, &io, &dio);
    const double Gp = dG / psi0, Ip = dI / psi0;
    const double rho = M * vpar / (q * B);
    const double D = Gs + io * Is + rho * (Gs * Ip - Is * Gp);
    const double a = io - rho * Gp, b = 1.0 + rho * Ip;
    out[0] = -W * (Gs * B_th - Is * B_ze) / D / psi0;
    out[1] = (Gs * W * B_psi + a * vpar * B) / D;
    out[2] = (b * vpar * B - Is * W * B_psi) / D;
    out[3] = -mu * B * (a * B_th + b * B_ze) / D;
    if (p->saw_on) out[0] = out[1] = out[2] = out[3] = NAN; /* the wave is defined on the vacuum model only */
    return;
  }
  if (!p->saw_on) {
    /* R1 (Boozer vacuum) */
    out[0] = -B_th * W / psi0;
    out[1] = B_psi * W + iota * vpar * B / G;
    out[2] = vpar * B / G;
    out[3] = -(iota * B_th + B_ze) * mu * B / G;
    return;
  }
  /* R2 (Boozer vacuum + shear Alfven wave): Phi = Phihat(s) sin(m th - n ze + w t),
     alpha from the ideal condition E_par = 0: d(alpha)/dt = -(iota Phi_th + Phi_ze)/G */
  const double diota = f->iota1;
  const double mm = (double)p->saw_m, nn = (double)p->saw_n, om = p->saw_omega;
  const double ds = s - p->saw_s0;
  const double Phihat = p->saw_Phi0 * exp(-ds * ds / p->saw_w2);
  const double dPhihat = Phihat * (-2.0 * ds / p->saw_w2);
  const double eta = mm * theta - nn * zeta + om * t;
  const double sn = sin(eta), cs = cos(eta);
  const double Phi = Phihat * sn;
  const double Phi_psi = dPhihat * sn / psi0;
  const double Phi_th = mm * Phihat * cs;
  const double Phi_ze = -nn * Phihat * cs;
  const double kpar = iota * mm - nn;
  const double al_th = -kpar * Phi_th / (om * G);
  const double al_t = -kpar * Phihat * cs / G;
  const double al_psi = -(diota * mm * Phi + kpar * dPhihat * sn) / (om * G) / psi0;
  const double psidot = -B_th * W + al_th * B * vpar - Phi_th;
  out[0] = psidot / psi0;
  out[1] = B_psi * W + (iota / G - al_psi) * vpar * B + Phi_psi;
  out[2] = vpar * B / G;
  out[3] = -(B / (G * M)) *
               (M * mu * (B_ze + al_th * B_psi * G + B_th * (iota - al_psi * G)) +
                q * (al_t * G + al_th * G * Phi_psi + (iota - al_psi * G) * Phi_th + Phi_ze)) +
           (vpar / B) * (B_th * Phi_psi - B_psi * Phi_th);
}

/* R3 (Cartesian vacuum guiding centre):
   xdot = vpar b + (M/(q|B|^3)) (vperp^2/2 + vpar^2) B x grad|B|,  vpardot = -mu b . grad|B|.
   fv holds cylindrical components on the (R,Z,phi) grid; they are rotated with the particle's own
   cos(phi) = x/R, sin(phi) = y/R. */
void orc_gc_cartesian(const orc_params *p, double mu, const double pos[3], double vpar,
                      const double fv[7], double out[4]) {
  const double M = p->mass, q = p->charge;
  const double R = sqrt(pos[0] * pos[0] + pos[1] * pos[1]);
  const double cph = pos[0] / R, sph = pos[1] / R;
  const double BR = fv[ORC_CY_BR], Bp = fv[ORC_CY_BPHI], BZ = fv[ORC_CY_BZ];
  const double gR = fv[ORC_CY_DB_DR], gp = fv[ORC_CY_DB_DPHI_R], gZ = fv[ORC_CY_DB_DZ];
  const double Bx = BR * cph - Bp * sph, By = BR * sph + Bp * cph, Bz = BZ;
  const double gx = gR * cph - gp * sph, gy = gR * sph + gp * cph, gz = gZ;
  const double modB = sqrt(BR * BR + Bp * Bp + BZ * BZ);
  const double vperp2 = 2.0 * mu * modB;
  const double coef = (M / (q * modB * modB * modB)) * (0.5 * vperp2 + vpar * vpar);
  const double cx = By * gz - Bz * gy, cy = Bz * gx - Bx * gz, cz = Bx * gy - By * gx;
  out[0] = vpar * Bx / modB + coef * cx;
  out[1] = vpar * By / modB + coef * cy;
  out[2] = vpar * Bz / modB + coef * cz;
  out[3] = -mu * (Bx * gx + By * gy + Bz * gz) / modB;
}

/* Stepped variables: Boozer (s cos th, s sin th, zeta, vpar); Cartesian as is. */
void orc_state_to_y(const orc_field *f, const double x[4], double y[4]) {
  if (f->coord == ORC_COORD_BOOZER) {
    y[0] = x[0] * cos(x[1]);
    y[1] = x[0] * sin(x[1]);
    y[2] = x[2];
    y[3] = x[3];
  } else {
    y[0] = x[0]; y[1] = x[1]; y[2] = x[2]; y[3] = x[3];
  }
}

void orc_y_to_state(const orc_field *f, const double y[4], double x[4]) {
  if (f->coord == ORC_COORD_BOOZER) {
    x[0] = sqrt(y[0] * y[0] + y[1] * y[1]);
    x[1] = atan2(y[1], y[0]);
    x[2] = y[2];
    x[3] = y[3];
  } else {
    x[0] = y[0]; x[1] = y[1]; x[2] = y[2]; x[3] = y[3];
  }
}

void orc_rhs(const orc_field *f, const orc_params *p, double mu, double t, const double y[4],
             double dy[4], double *fv_out) {
  double fv[16], d[4];
  if (f->coord == ORC_COORD_BOOZER) {
    const double s = sqrt(y[0] * y[0] + y[1] * y[1]);
    const double theta = atan2(y[1], y[0]);
    const double x[3] = {s, theta, y[2]};
    if (f->nquant == 1 && !f->analytic) {
      /* reading R1c (derivative-of-interpolant mode): only |B| is tabulated, its derivatives are those of its
         interpolant */
      orc_tricubic_grad(f, x, 0, &fv[0], &fv[1]);
    } else {
      orc_tricubic(f, x, fv);
    }
    orc_gc_boozer(f, p, mu, t, s, theta, y[2], y[3], fv, d);
    /* d/dt (s cos th, s sin th) with cos th = y0/s, sin th = y1/s */
    const double c = (s > 0.0) ? y[0] / s : 1.0, sn = (s > 0.0) ? y[1] / s : 0.0;
    dy[0] = d[0] * c - d[1] * y[1];
    dy[1] = d[0] * sn + d[1] * y[0];
    dy[2] = d[2];
    dy[3] = d[3];
  } else {
    const double R = sqrt(y[0] * y[0] + y[1] * y[1]);
    const double x[3] = {R, y[2], atan2(y[1], y[0])};
    orc_tricubic(f, x, fv);
    orc_gc_cartesian(p, mu, y, y[3], fv, dy);
  }
  if (fv_out) memcpy(fv_out, fv, sizeof(double) * (size_t)(f->nquant == 1 ? 4 : f->nquant));
}

/* ------------------------------------------------------------------------------------------
 * Dormand-Prince 5(4) (ref [10] PAPER.md:164), Boost-odeint-style controller.
 * ---------------------------------------------------------------------------------------- */
static const double DP_C[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
static const double DP_A[7][7] = {
    {0},
    {1.0 / 5.0},
    {3.0 / 40.0, 9.0 / 40.0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
static const double DP_B[7] = {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0,
                               -2187.0 / 6784.0, 11.0 / 84.0, 0.0};
/* b - bhat */
static const double DP_E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0,
                               -17253.0 / 339200.0, 22.0 / 525.0, -1.0 / 40.0};

void orc_dp5_tableau(double c[7], double a[7][7], double b[7], double e[7]) {
  memcpy(c, DP_C, sizeof(DP_C));
  memcpy(a, DP_A, sizeof(DP_A));
  memcpy(b, DP_B, sizeof(DP_B));
  memcpy(e, DP_E, sizeof(DP_E));
}

#define ORC_MAXN 8

void orc_dp5_attempt(orc_ode_fn fn, void *ctx, int n, double t, const double *y, const double *k1,
                     double h, double *ynew, double *k7, double *err, double *kall) {
  double k[7][ORC_MAXN], ys[ORC_MAXN];
  for (int i = 0; i < n; ++i) k[0][i] = k1[i];
  for (int st = 1; st < 7; ++st) {
    for (int i = 0; i < n; ++i) {
      double acc = 0.0;
      for (int j = 0; j < st; ++j) acc += DP_A[st][j] * k[j][i];
      ys[i] = y[i] + h * acc;
    }
    fn(ctx, t + DP_C[st] * h, ys, k[st]);
  }
  /* stage 7 is evaluated at the new state (a_7j = b_j): first-same-as-last */
  for (int i = 0; i < n; ++i) {
    ynew[i] = ys[i];
    k7[i] = k[6][i];
    double e = 0.0;
    for (int j = 0; j < 7; ++j) e += DP_E[j] * k[j][i];
    err[i] = h * e;
  }
  if (kall)
    for (int j = 0; j < 7; ++j)
      for (int i = 0; i < n; ++i) kall[j * n + i] = k[j][i];
}

/* PAPER.md:85 Eq. 4: error = max_i |e_i| / (atol_i c_i + rtol_i (|x_i| + dt |xdot_i|)),
   x and xdot taken at the start of the step (Boost default error checker). */
double orc_error_ratio(int n, const double *err, const double *y, const double *k1, double h,
                       double rtol, double atol, const double *cscale) {
  double r = 0.0;
  for (int i = 0; i < n; ++i) {
    const double den = atol * cscale[i] + rtol * (fabs(y[i]) + fabs(h) * fabs(k1[i]));
    const double v = fabs(err[i]) / den;
    if (v != v) return v; /* a non-finite component makes the step a rejection */
    if (v > r) r = v;
  }
  return r;
}

/* Boost odeint default step adjuster for dopri5 (stepper order 5, error order 4):
   r > 1  : reject, dt <- dt * max(0.9 r^(-1/3), 1/5)
   r < 0.5: accept, dt <- dt * 0.9 max(r, 5^-5)^(-1/5)   (growth <= 4.5x)
   else   : accept, dt unchanged.  dt never exceeds dtmax. */
double orc_controller(double h, double r, double dtmax, int *accepted) {
  double dt = h;
  if (!(r <= 1.0)) {
    *accepted = 0;
    double fac = 0.9 * pow(r, -1.0 / 3.0);
    if (!(fac >= 0.2)) fac = 0.2;
    dt = h * fac;
  } else {
    *accepted = 1;
    if (r < 0.5) {
      double rr = r;
      const double floor5 = 1.0 / 3125.0;
      if (rr < floor5) rr = floor5;
      dt = h * 0.9 * pow(rr, -1.0 / 5.0);
    }
  }
  if (dtmax > 0.0 && dt > dtmax) dt = dtmax;
  return dt;
}

/* ------------------------------------------------------------------------------------------
 * Whole tracer
 * ---------------------------------------------------------------------------------------- */
double orc_vtotal(const orc_params *p) { return sqrt(2.0 * p->energy / p->mass); }

/* DESIGN.md reading S3 (paper silent): dtmax = (pi/2) L / v_total, dt0 = 1e-3 dtmax,
   L = |G0| / |B|(first node) for Boozer, L = hi[0] (R_max) for the cylindrical grid. */
void orc_default_steps(const orc_field *f, const orc_params *p, double *dt0, double *dtmax) {
  double L;
  if (f->coord == ORC_COORD_BOOZER) {
    const double Bref = f->nodes ? fabs(f->nodes[0]) : 1.0;
    L = fabs(f->G_nodes ? f->G_nodes[0] : f->G0) / Bref; /* non-vacuum: G on the axis */
  } else {
    L = f->hi[0];
  }
  double mx = p->dtmax > 0.0 ? p->dtmax : 0.5 * ORC_PI * L / orc_vtotal(p);
  double d0 = p->dt0 > 0.0 ? p->dt0 : 1e-3 * mx;
  if (d0 > mx) d0 = mx;
  *dt0 = d0;
  *dtmax = mx;
}

static double orc_modB_at(const orc_field *f, const double y[4], double *psi_out) {
  double fv[16];
  if (f->coord == ORC_COORD_BOOZER) {
    const double s = sqrt(y[0] * y[0] + y[1] * y[1]);
    const double x[3] = {s, atan2(y[1], y[0]), y[2]};
    orc_tricubic(f, x, fv);
    if (psi_out) *psi_out = s;
    return fv[ORC_BZ_MODB];
  }
  const double R = sqrt(y[0] * y[0] + y[1] * y[1]);
  const double x[3] = {R, y[2], atan2(y[1], y[0])};
  orc_tricubic(f, x, fv);
  if (psi_out) *psi_out = fv[ORC_CY_PSI];
  return sqrt(fv[ORC_CY_BR] * fv[ORC_CY_BR] + fv[ORC_CY_BPHI] * fv[ORC_CY_BPHI] +
              fv[ORC_CY_BZ] * fv[ORC_CY_BZ]);
}

/* mu = (v^2 - vpar^2) / (2 B(x0)) per unit mass, B from the tabulated field */
double orc_mu_init(const orc_field *f, const orc_params *p, const double x[4]) {
  double y[4];
  orc_state_to_y(f, x, y);
  const double B = orc_modB_at(f, y, NULL);
  const double v = orc_vtotal(p);
  return (v * v - x[3] * x[3]) / (2.0 * B);
}

/* loss level: Boozer s >= 1; Cartesian: interpolated level function psi >= psi_edge */
static int orc_is_lost(const orc_field *f, const double y[4]) {
  if (f->coord == ORC_COORD_BOOZER) return sqrt(y[0] * y[0] + y[1] * y[1]) >= 1.0;
  double psi;
  (void)orc_modB_at(f, y, &psi);
  return psi >= f->psi0;
}

/* DESIGN.md reading S5b.  The step from (y0, derivative k0) to (y1, derivative k1) of length h crossed the loss
 * boundary: orc_is_lost(y0) is false, orc_is_lost(y1) true.  The stepped variables are interpolated inside the step
 * by the cubic Hermite polynomial of the two end states and end derivatives (both are at hand: k1 is the step's
 * seventh stage, first-same-as-last), theta in [0,1]:
 *   y(theta) = (2 th^3 - 3 th^2 + 1) y0 + (th^3 - 2 th^2 + th) h k0 + (-2 th^3 + 3 th^2) y1 + (th^3 - th^2) h k1.
 * The loss time is t + theta* h with theta* found by 48 bisections on "orc_is_lost(y(theta))" from [0,1]: the
 * smallest theta the bisection observes beyond the boundary; the returned state is y(theta*). */
void orc_hermite_state(const double y0[4], const double k0[4], const double y1[4], const double k1[4], double h,
                       double theta, double y[4]) {
  const double t2 = theta * theta, t3 = t2 * theta;
  const double h00 = 2.0 * t3 - 3.0 * t2 + 1.0, h10 = t3 - 2.0 * t2 + theta;
  const double h01 = -2.0 * t3 + 3.0 * t2, h11 = t3 - t2;
  for (int i = 0; i < 4; ++i) y[i] = h00 * y0[i] + h10 * h * k0[i] + h01 * y1[i] + h11 * h * k1[i];
}

double orc_loss_refine(const orc_field *f, const double y0[4], const double k0[4], const double y1[4],
                       const double k1[4], double h, double y[4]) {
  double lo = 0.0, hi = 1.0;
  for (int it = 0; it < 48; ++it) {
    const double mid = 0.5 * (lo + hi);
    double ym[4];
    orc_hermite_state(y0, k0, y1, k1, h, mid, ym);
    if (orc_is_lost(f, ym)) hi = mid;
    else lo = mid;
  }
  orc_hermite_state(y0, k0, y1, k1, h, hi, y);
  return hi;
}

typedef struct {
  const orc_field *f;
  const orc_params *p;
  double mu;
} orc_rhs_ctx;

static void orc_rhs_cb(void *ctx, double t, const double *y, double *dy) {
  const orc_rhs_ctx *c = (const orc_rhs_ctx *)ctx;
  orc_rhs(c->f, c->p, c->mu, t, y, dy, NULL);
}

static void orc_trace_one(const orc_field *f, const orc_params *p, const double x0[4],
                          double xf[4], double *tstop, int32_t *status, uint32_t *nacc_o,
                          uint32_t *nrej_o, double *traj, int64_t maxrec, int64_t *nrec_o) {
  double y[4], k1[4], ynew[4], k7[4], err[4];
  const double vtot = orc_vtotal(p);
  const double cscale[4] = {1.0, 1.0, 1.0, vtot};
  double dt, dtmax;
  orc_default_steps(f, p, &dt, &dtmax);
  const int maxrej = p->max_consecutive_rejects > 0 ? p->max_consecutive_rejects : 500;
  uint32_t nacc = 0, nrej = 0;
  int64_t nrec = 0;
  int consecutive = 0;
  double t = 0.0;
  int32_t st = 0;

  orc_state_to_y(f, x0, y);
  if (orc_is_lost(f, y)) { /* already outside: returned unchanged with t_stop = 0 */
    for (int i = 0; i < 4; ++i) xf[i] = x0[i];
    *tstop = 0.0;
    *status = 1;
    if (nacc_o) *nacc_o = 0;
    if (nrej_o) *nrej_o = 0;
    if (nrec_o) *nrec_o = 0;
    return;
  }
  orc_rhs_ctx ctx = {f, p, orc_mu_init(f, p, x0)};
  orc_rhs_cb(&ctx, t, y, k1);
  if (traj && nrec < maxrec) {
    double xs[4];
    orc_y_to_state(f, y, xs);
    traj[nrec * 5] = t;
    for (int i = 0; i < 4; ++i) traj[nrec * 5 + 1 + i] = xs[i];
    ++nrec;
  }
  if (!(p->T > 0.0)) {
    st = 0;
  } else
    for (;;) {
      if (p->max_steps > 0 && (int64_t)nacc + (int64_t)nrej >= p->max_steps) { st = 3; break; }
      /* DESIGN.md reading S4: the last step lands exactly on T */
      const double rem = p->T - t;
      const int clamped = !(dt < rem);
      const double h = clamped ? rem : dt;
      orc_dp5_attempt(orc_rhs_cb, &ctx, 4, t, y, k1, h, ynew, k7, err, NULL);
      const double r = orc_error_ratio(4, err, y, k1, h, p->rtol, p->atol, cscale);
      int accepted;
      const double dtn = orc_controller(h, r, dtmax, &accepted);
      if (!accepted) {
        ++nrej;
        dt = dtn;
        if (++consecutive >= maxrej) { st = 2; break; } /* reading S6 */
        continue;
      }
      consecutive = 0;
      ++nacc;
      if (p->loss_time_mode == 1 && orc_is_lost(f, ynew)) { /* reading S5b: the loss time inside this step */
        double yl[4];
        const double theta = orc_loss_refine(f, y, k1, ynew, k7, h, yl);
        t = t + theta * h;
        for (int i = 0; i < 4; ++i) y[i] = yl[i];
        if (traj && nrec < maxrec) {
          double xs[4];
          orc_y_to_state(f, y, xs);
          traj[nrec * 5] = t;
          for (int i = 0; i < 4; ++i) traj[nrec * 5 + 1 + i] = xs[i];
          ++nrec;
        }
        st = 1;
        break;
      }
      t = clamped ? p->T : t + h;
      if (!clamped) dt = dtn; /* the clamp does not shrink the controller's memory */
      for (int i = 0; i < 4; ++i) { y[i] = ynew[i]; k1[i] = k7[i]; }
      if (traj && nrec < maxrec) {
        double xs[4];
        orc_y_to_state(f, y, xs);
        traj[nrec * 5] = t;
        for (int i = 0; i < 4; ++i) traj[nrec * 5 + 1 + i] = xs[i];
        ++nrec;
      }
      /* reading S5: loss first, then T */
      if (orc_is_lost(f, y)) { st = 1; break; }
      if (t >= p->T) { st = 0; break; }
    }
  orc_y_to_state(f, y, xf);
  *tstop = t;
  *status = st;
  if (nacc_o) *nacc_o = nacc;
  if (nrej_o) *nrej_o = nrej;
  if (nrec_o) *nrec_o = nrec;
}

void orc_trace(const orc_field *f, const orc_params *p, int64_t n, const double *x0, double *xf,
               double *tstop, int32_t *status, uint32_t *nacc, uint32_t *nrej, int nthreads) {
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
  (void)nthreads;
#endif
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
  for (int64_t i = 0; i < n; ++i) {
    double a[4] = {x0[i], x0[n + i], x0[2 * n + i], x0[3 * n + i]}, b[4], ts;
    int32_t st;
    uint32_t na, nr;
    orc_trace_one(f, p, a, b, &ts, &st, &na, &nr, NULL, 0, NULL);
    for (int c = 0; c < 4; ++c) xf[c * n + i] = b[c];
    tstop[i] = ts;
    status[i] = st;
    if (nacc) nacc[i] = na;
    if (nrej) nrej[i] = nr;
  }
}

int64_t orc_trace_record(const orc_field *f, const orc_params *p, const double x0[4], double *traj,
                         int64_t maxrec, double *tstop, int32_t *status) {
  double xf[4];
  int64_t nrec = 0;
  orc_trace_one(f, p, x0, xf, tstop, status, NULL, NULL, traj, maxrec, &nrec);
  return nrec;
}

int64_t orc_trace_scripted(const orc_field *f, const orc_params *p, const double x0[4], int64_t nsteps,
                           const double *h, double xf[4], double *tstop, int32_t *status, double *r) {
  double y[4], k1[4], ynew[4], k7[4], err[4];
  const double cscale[4] = {1.0, 1.0, 1.0, orc_vtotal(p)};
  double t = 0.0;
  int64_t taken = 0;
  int32_t st = 0;
  orc_state_to_y(f, x0, y);
  if (orc_is_lost(f, y)) {
    for (int i = 0; i < 4; ++i) xf[i] = x0[i];
    *tstop = 0.0;
    *status = 1;
    return 0;
  }
  orc_rhs_ctx ctx = {f, p, orc_mu_init(f, p, x0)};
  orc_rhs_cb(&ctx, t, y, k1);
  while (taken < nsteps && h[taken] > 0.0) {
    const double hh = h[taken];
    orc_dp5_attempt(orc_rhs_cb, &ctx, 4, t, y, k1, hh, ynew, k7, err, NULL);
    if (r) r[taken] = orc_error_ratio(4, err, y, k1, hh, p->rtol, p->atol, cscale);
    ++taken;
    if (p->loss_time_mode == 1 && orc_is_lost(f, ynew)) { /* reading S5b */
      double yl[4];
      const double theta = orc_loss_refine(f, y, k1, ynew, k7, hh, yl);
      t = t + theta * hh;
      for (int i = 0; i < 4; ++i) y[i] = yl[i];
      st = 1;
      break;
    }
    t = t + hh;
    for (int i = 0; i < 4; ++i) { y[i] = ynew[i]; k1[i] = k7[i]; }
    if (orc_is_lost(f, y)) { st = 1; break; }
  }
  orc_y_to_state(f, y, xf);
  *tstop = t;
  *status = st;
  return taken;
}

void orc_step_once(const orc_field *f, const orc_params *p, const double x[4], double t, double h,
                   double xnew[4], double *errratio, double *k) {
  double y[4], k1[4], ynew[4], k7[4], err[4];
  const double cscale[4] = {1.0, 1.0, 1.0, orc_vtotal(p)};
  orc_state_to_y(f, x, y);
  orc_rhs_ctx ctx = {f, p, orc_mu_init(f, p, x)};
  orc_rhs_cb(&ctx, t, y, k1);
  orc_dp5_attempt(orc_rhs_cb, &ctx, 4, t, y, k1, h, ynew, k7, err, k);
  *errratio = orc_error_ratio(4, err, y, k1, h, p->rtol, p->atol, cscale);
  orc_y_to_state(f, ynew, xnew);
}

/* PAPER.md:29 Eq. 2: phi_hat = (1/n) sum g(Y_i); standard error sqrt((sum g^2/n - phi^2)/(n-1)) */
void orc_estimate(int g_kind, int64_t n, const int32_t *status, const double *tstop,
                  const double *g_user, double out[3]) {
  double sum = 0.0, sum2 = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    double g;
    if (g_kind == 0) g = (status[i] == 1) ? 1.0 : 0.0;
    else if (g_kind == 1) g = tstop[i];
    else g = g_user[i];
    sum += g;
    sum2 += g * g;
  }
  const double mean = n > 0 ? sum / (double)n : 0.0;
  double var = n > 1 ? (sum2 / (double)n - mean * mean) / (double)(n - 1) : 0.0;
  if (var < 0.0) var = 0.0;
  out[0] = mean;
  out[1] = sqrt(var);
  out[2] = sum;
}

/* ---- other measurements g ("Similar functions g can be chosen to calculate energy loss ..., wall-loads
 * from alpha particles"; readings G2, G3).  Both look at the END state of a trace only. ---- */

/* Reading G2, lost energy: g_i = 1[lost] E_i / E_0 with the guiding-centre energy per unit mass at the exit point,
 * E_i = vpar^2 / 2 + mu |B|(x_f) (mu = v_perp^2 / (2B) per unit mass), |B| from the tabulated field, and
 * E_0 = v_total^2 / 2 the birth energy every particle shares.  Its mean (Eq. 2) is the fraction of the
 * alpha power that leaves with lost particles; with a wave E_i differs from E_0. */
void orc_lost_energy(const orc_field *f, const orc_params *p, int64_t n, const double *xf /*[4][n]*/,
                     const double *mu /*[n]*/, const int32_t *status, double *g /*[n]*/) {
  const double v = orc_vtotal(p);
  const double E0 = 0.5 * v * v;
  for (int64_t i = 0; i < n; ++i) {
    if (status[i] != 1) { g[i] = 0.0; continue; }
    const double x[4] = {xf[i], xf[n + i], xf[2 * n + i], xf[3 * n + i]};
    double y[4];
    orc_state_to_y(f, x, y);
    const double B = orc_modB_at(f, y, NULL);
    g[i] = (0.5 * x[3] * x[3] + mu[i] * B) / E0;
  }
}

/* one histogram bin: u = (a - lo) / span, reduced to [0, 1) when periodic, bin = floor(u nb) clamped to [0, nb-1] */
static int orc_bin(double a, double lo, double span, int periodic, int nb) {
  double u = (a - lo) / span;
  if (periodic) u = u - floor(u);
  int b = (int)floor(u * (double)nb);
  if (b < 0) b = 0;
  if (b > nb - 1) b = nb - 1;
  return b;
}

/* Reading G3, wall load: the number of lost particles per bin of the exit point, hist[nb0][nb1].
 * Boozer: (theta over [0, 2 pi), zeta over one field period [lo2, hi2)), both periodic.
 * Cylindrical: (phi = atan2(y, x) over one field period [lo2, hi2), periodic; Z over [lo1, hi1], clamped). */
void orc_exit_histogram(const orc_field *f, int64_t n, const double *xf /*[4][n]*/, const int32_t *status,
                        int nb0, int nb1, int64_t *hist /*[nb0][nb1]*/) {
  for (int k = 0; k < nb0 * nb1; ++k) hist[k] = 0;
  for (int64_t i = 0; i < n; ++i) {
    if (status[i] != 1) continue;
    int b0, b1;
    if (f->coord == ORC_COORD_BOOZER) {
      b0 = orc_bin(xf[n + i], f->lo[1], f->hi[1] - f->lo[1], 1, nb0);
      b1 = orc_bin(xf[2 * n + i], f->lo[2], f->hi[2] - f->lo[2], 1, nb1);
    } else {
      b0 = orc_bin(atan2(xf[n + i], xf[i]), f->lo[2], f->hi[2] - f->lo[2], 1, nb0);
      b1 = orc_bin(xf[2 * n + i], f->lo[1], f->hi[1] - f->lo[1], 0, nb1);
    }
    hist[b0 * nb1 + b1] += 1;
  }
}

int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
