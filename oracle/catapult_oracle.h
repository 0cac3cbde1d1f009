/*
 * CATAPULT oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU restatement of what the hot path of
 * arxiv/paper_2604_07617 (CATAPULT) computes, written from PAPER.md and the
 * readings listed in DESIGN.md.  It shares no code with the CUDA library under
 * paper_2604_07617_b200/csrc and is only ever called from tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * Every function cites the passage of PAPER.md it follows.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   orc_lagrange4 / orc_tricubic : node reproduction, partition of unity,
 *       exact reproduction of tricubic polynomials (also extrapolated),
 *       face continuity, scipy BarycentricInterpolator special case.
 *   orc_field_build              : brute-force index identity.
 *   DP5 tableau / orc_dp5_attempt: row sums, order-5 convergence, scipy RK45
 *       single step and error vector.
 *   controller                   : closed-form table of r -> dt.
 *   orc_gc_boozer (R1,R2)        : Euler-Lagrange equations of PAPER.md Eq. 3
 *       derived independently with sympy; B=B(s) closed form; energy; P_zeta;
 *       n*H - omega*P_zeta with a wave.
 *   orc_gc_cartesian (R3)        : pure toroidal field closed form; energy;
 *       P_phi in an axisymmetric field.
 *   orc_default_steps            : hand values of reading S3 (9.37e-7 s for config 0, |G|/|B|(node 0) and R_max
 *       retyped from the constants), explicit values win, dt0 clamped to dtmax.
 *   orc_trace                    : brute-force fixed-step RK4 on a tiny ensemble.
 *   orc_estimate                 : numpy.mean.
 *   orc_lost_energy (G2)         : hand value from the closed-form |B| at a grid node; energy conservation in a
 *       static field (g = 1 for every lost particle, interpolation-limited); 0 for particles that are not lost.
 *   orc_exit_histogram (G3)      : numpy.histogram2d on independently reduced angles; hand-placed particles.
 * Parity unpinned: absolute loss fractions of the five configs (nothing in the
 * paper fixes them).
 */
#ifndef CATAPULT_ORACLE_H
#define CATAPULT_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_COORD_BOOZER 0 /* (s, theta, zeta) grid, state (s,theta,zeta,vpar)   */
#define ORC_COORD_CYL    1 /* (R, Z, phi) grid,     state (x,y,z,vpar) Cartesian */

/* column order of the gridded quantities (PAPER.md:45 for Boozer vacuum) */
#define ORC_BZ_MODB   0
#define ORC_BZ_DB_DS  1
#define ORC_BZ_DB_DTH 2
#define ORC_BZ_DB_DZE 3
#define ORC_CY_BR     0
#define ORC_CY_BPHI   1
#define ORC_CY_BZ     2
#define ORC_CY_DB_DR  3
#define ORC_CY_DB_DPHI_R 4 /* (1/R) d|B|/dphi */
#define ORC_CY_DB_DZ  5
#define ORC_CY_PSI    6    /* loss level function */

/* analytic-field hook used ONLY by pins: replaces the table lookup.
   x = (s,theta,zeta) or (R,Z,phi), unreduced; out[nquant]. */
typedef void (*orc_analytic_fn)(void *ctx, const double *x, double *out);

typedef struct {
  int32_t coord;
  int32_t ncell[3]; /* cells per dimension, slowest -> fastest  */
  int32_t nfp;
  int32_t nquant;   /* m                                                     */
  double lo[3], hi[3];
  const double *nodes; /* [m][3*ncell0+1][3*ncell1+1][3*ncell2+1] unique nodes */
  double G0, I0;       /* Boozer covariant components (constants; vacuum: I0 = 0) */
  double iota0, iota1; /* iota(s) = iota0 + iota1*s                           */
  double psi0;         /* Boozer: toroidal flux/2pi at s=1; cyl: psi_edge      */
  orc_analytic_fn analytic; /* NULL => tables */
  void *analytic_ctx;
  /* non-vacuum Boozer ("vacuum, finite beta, etc."; reading R1b): G(s), I(s), iota(s) on the
     3*ncell[0]+1 unique s-nodes of the grid (all three or none; NULL => the scalars G0, I0 = 0 and the linear law) */
  const double *G_nodes, *I_nodes, *iota_nodes;
} orc_field;

typedef struct {
  double mass, charge, energy; /* shared by all particles */
  double T, rtol, atol;        /* PAPER.md:85 Eq. 4 */
  double dt0, dtmax;           /* <=0 => defaults (reading S3) */
  int64_t max_steps;           /* 0 => unlimited */
  int32_t max_consecutive_rejects; /* 0 => 500 */
  int32_t saw_on, saw_m, saw_n;
  double saw_Phi0, saw_s0, saw_w2, saw_omega; /* Phi0 exp(-(s-s0)^2/w2) sin(m th - n ze + omega t) */
  int32_t loss_time_mode;      /* 0: end of the step that crossed (reading S5); 1: root inside it (reading S5b) */
  int32_t reserved_;
} orc_params;

/* ---- other measurements g (readings G2, G3) ---- */
void orc_lost_energy(const orc_field *f, const orc_params *p, int64_t n, const double *xf, const double *mu,
                     const int32_t *status, double *g);
void orc_exit_histogram(const orc_field *f, int64_t n, const double *xf, const int32_t *status, int nb0, int nb1,
                        int64_t *hist);

/* ---- loss time inside the last step (reading S5b; tau, "the first time the particle
 * is observed beyond the boundary", sharpened) ---- */
void orc_hermite_state(const double y0[4], const double k0[4], const double y1[4], const double k1[4], double h,
                       double theta, double y[4]);
double orc_loss_refine(const orc_field *f, const double y0[4], const double k0[4], const double y1[4],
                       const double k1[4], double h, double y[4]);

/* ---- 1-D profiles on the s-nodes: value and d/ds by the same piecewise cubic as the tables ---- */
void orc_dlagrange4(double u, double dL[4]);
void orc_profile(const orc_field *f, const double *nodes, double s, double *val, double *dval_ds);

/* ---- tricubic ---- */
void orc_lagrange4(double u, double L[4]);
void orc_locate(const orc_field *f, const double x[3], int32_t cell[3], double u[3]);
void orc_tricubic(const orc_field *f, const double x[3], double *out /*[m]*/);
/* value and gradient (with respect to the three grid coordinates) of quantity q's interpolant: the local tricubic of
   PAPER.md:47-53 differentiated (reading R1c, the derivative-of-interpolant mode) */
void orc_tricubic_grad(const orc_field *f, const double x[3], int q, double *val, double grad[3]);
void orc_tricubic_many(const orc_field *f, int64_t npts, const double *pts /*[3][npts]*/,
                       double *out /*[m][npts]*/);
/* paper's stored layout D1: out[((cell*64)+node)*m + q], cell and node ordered dim0,dim1,dim2
   slowest->fastest */
void orc_field_build(const orc_field *f, double *out);

/* ---- right-hand sides (Eq. 3; R1-R3) ---- */
/* physics only: field values in, (sdot, thetadot, zetadot, vpardot) out. */
void orc_gc_boozer(const orc_field *f, const orc_params *p, double mu, double t,
                   double s, double theta, double zeta, double vpar,
                   const double fv[4] /* B, dB/ds, dB/dtheta, dB/dzeta */,
                   double out[4]);
void orc_gc_cartesian(const orc_params *p, double mu, const double pos[3], double vpar,
                      const double fv[7], double out[4]);
/* full RHS in the stepped variables: Boozer y=(s cos th, s sin th, zeta, vpar),
   Cartesian y=(x,y,z,vpar).  fv_out (may be NULL) receives the interpolated columns. */
void orc_rhs(const orc_field *f, const orc_params *p, double mu, double t, const double y[4],
             double dy[4], double *fv_out);

/* ---- DP5(4) (Dormand & Prince 1980) ---- */
typedef void (*orc_ode_fn)(void *ctx, double t, const double *y, double *dy);
/* tableau access for pins */
void orc_dp5_tableau(double c[7], double a[7][7], double b[7], double e[7]);
/* one attempted step of size h from (t,y) with k1=f(t,y): ynew, k7=f(t+h,ynew), err=h*sum e_i k_i,
   kall (may be NULL) gets all 7 stage derivatives [7][n] */
void orc_dp5_attempt(orc_ode_fn fn, void *ctx, int n, double t, const double *y, const double *k1,
                     double h, double *ynew, double *k7, double *err, double *kall);
/* Eq. 4 with scale vector c */
double orc_error_ratio(int n, const double *err, const double *y, const double *k1, double h,
                       double rtol, double atol, const double *cscale);
/* Boost-rule controller: returns the next dt given the attempted h and ratio r;
   *accepted = (r <= 1) */
double orc_controller(double h, double r, double dtmax, int *accepted);

/* ---- whole tracer ---- */
double orc_vtotal(const orc_params *p);
void orc_default_steps(const orc_field *f, const orc_params *p, double *dt0, double *dtmax);
/* converts API state (s,th,ze,vpar)/(x,y,z,vpar) to stepped variables and back */
void orc_state_to_y(const orc_field *f, const double x[4], double y[4]);
void orc_y_to_state(const orc_field *f, const double y[4], double x[4]);
double orc_mu_init(const orc_field *f, const orc_params *p, const double x[4]);

/* status: 0 reached T, 1 lost, 2 stalled, 3 max_steps */
void orc_trace(const orc_field *f, const orc_params *p, int64_t n, const double *x0 /*[4][n]*/,
               double *xf /*[4][n]*/, double *tstop, int32_t *status, uint32_t *nacc,
               uint32_t *nrej, int nthreads);
/* single attempted step from API state x at time t with step h (test hook twin of
   catapult_step_once): xnew (API coords), errratio, k[7][4] */
void orc_step_once(const orc_field *f, const orc_params *p, const double x[4], double t, double h,
                   double xnew[4], double *errratio, double *k /*[7][4]*/);
/* trace one particle recording every accepted state: traj[(i)*5 + (t,y0..y3 API coords)] up to maxrec */
int64_t orc_trace_record(const orc_field *f, const orc_params *p, const double x0[4], double *traj,
                         int64_t maxrec, double *tstop, int32_t *status);

/* scripted replay of one particle (twin of catapult_trace_scripted): takes the step sizes h[0..nsteps)
   one after the other from t=0, every step accepted whatever its error ratio (written to r[i]); stops
   at the first h <= 0, after nsteps steps, or when an end state is beyond the loss boundary.  Returns
   the number of steps taken; status 1 if lost else 0.  Lets a test walk another run's accepted-step
   sequence without any accept/reject decision in between. */
int64_t orc_trace_scripted(const orc_field *f, const orc_params *p, const double x0[4], int64_t nsteps,
                           const double *h, double xf[4], double *tstop, int32_t *status, double *r);

/* ---- estimator (Eq. 2) ---- */
/* g_kind 0: 1[status==1], 1: tstop, 2: user array.  out = {mean, standard error, sum} */
void orc_estimate(int g_kind, int64_t n, const int32_t *status, const double *tstop,
                  const double *g_user, double out[3]);

int orc_max_threads(void);

#ifdef __cplusplus
}
#endif
#endif
