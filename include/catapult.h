/*
 * catapult.h -- C-ABI of the B200-native CATAPULT hot path (arxiv/paper_2604_07617).
 *
 * What it computes (PAPER.md = the paper's text; DESIGN.md lists every reading of a silent point):
 *   per-particle tracing of the Littlejohn guiding-centre equations (Eq. 3) in
 *   Boozer (s,theta,zeta,vpar) and Cartesian (x,y,z,vpar) form with Dormand-Prince 5(4) adaptive
 *   steps (Eq. 4 at PAPER.md:85), every stage evaluating a local tricubic interpolant
 *   of gridded field quantities, stopping at the loss boundary or at T
 *   (PAPER.md:57-59), and the Monte-Carlo estimate of Eq. 2.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers; all are owned by the caller,
 *     the library never frees them.  `stream` is a cudaStream_t passed as void* (NULL = default
 *     stream).  All work runs on the device that is current when the call is made.
 *   - Every call returns a catapult_status; no exception crosses the boundary;
 *     catapult_last_error() returns a thread-local message for the last failing call.
 *   - Calls validate their arguments synchronously, enqueue work on `stream` and do not
 *     synchronise (device memory they need is allocated and freed stream-ordered), except: the
 *     *_host variants and catapult_estimate with a non-NULL h_out, which return after their
 *     results are in host memory, catapult_field_destroy, which waits for ALL work on the field's
 *     device (cudaDeviceSynchronize: traces of the field may be running on any stream) before it
 *     frees the tables, so a field may be destroyed right after an asynchronous call that uses it,
 *     and catapult_release_host_cache (cudaFree of the calling thread's staging slab, which came
 *     from cudaMalloc and therefore waits for the device).
 *     A field may be used on any stream: every call that reads its tables is ordered after the
 *     build by an event the build recorded.
 *   - There is no CPU fallback anywhere: without a CUDA device every compute call fails with
 *     CATAPULT_ECUDA.
 *   - Particle arrays are structure-of-arrays: x[4][n] means component c of particle i at
 *     x[c*n + i].  Boozer state = (s, theta, zeta, vpar); Cartesian state = (x, y, z, vpar).
 */
#ifndef CATAPULT_H
#define CATAPULT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  CATAPULT_OK = 0,
  CATAPULT_EINVAL = 1,       /* bad argument (NULL required pointer, n<0, ncell<1, non-finite T/rtol/atol ...) */
  CATAPULT_ENOMEM = 2,       /* device or host allocation failed */
  CATAPULT_ECUDA = 3,        /* CUDA runtime error (message in catapult_last_error) */
  CATAPULT_EUNSUPPORTED = 4  /* valid but not built (e.g. a non-canonical column order, the wave on a non-vacuum field) */
} catapult_status;

#define CATAPULT_COORD_BOOZER 0 /* grid (s,theta,zeta); particles (s,theta,zeta,vpar)            */
#define CATAPULT_COORD_CYL 1    /* grid (R,Z,phi); particles (x,y,z,vpar)       */

/* Column (quantity) order of the gridded data.
   Boozer vacuum: |B|, d|B|/ds, d|B|/dtheta, d|B|/dzeta            -> nquant = 4
   Cylindrical grid (R3): B_R, B_phi, B_Z, d|B|/dR, (1/R) d|B|/dphi, d|B|/dZ,
                                    psi (loss level function)        -> nquant = 7 */
#define CATAPULT_NQUANT_BOOZER 4
/* Boozer, derivative-of-interpolant mode (R1c): only |B| is tabulated (nquant = 1, one 512-byte block per
   cell instead of four); d|B|/ds, d|B|/dtheta, d|B|/dzeta are the derivatives of its local tricubic.  The right-hand
   side then jumps at cell faces: more attempts are rejected and more steps are needed than with tabulated
   derivative columns. */
#define CATAPULT_NQUANT_BOOZER_DOI 1
#define CATAPULT_NQUANT_CYL 7

/* semantic tags of the columns (catapult_field_desc.quant).  All sixteen entries zero = the canonical
   order above; otherwise quant[0..nquant) must spell out that same order (other orders: EUNSUPPORTED) */
#define CATAPULT_Q_MODB 1
#define CATAPULT_Q_DMODB_DS 2
#define CATAPULT_Q_DMODB_DTHETA 3
#define CATAPULT_Q_DMODB_DZETA 4
#define CATAPULT_Q_B_R 5
#define CATAPULT_Q_B_PHI 6
#define CATAPULT_Q_B_Z 7
#define CATAPULT_Q_DMODB_DR 8
#define CATAPULT_Q_DMODB_DPHI_OVER_R 9
#define CATAPULT_Q_DMODB_DZ 10
#define CATAPULT_Q_PSI_LEVEL 11

/* particle status */
#define CATAPULT_ST_REACHED_T 0
#define CATAPULT_ST_LOST 1      /* s >= 1 (Boozer) or psi >= psi_edge (Cartesian) */
#define CATAPULT_ST_STALLED 2   /* max_consecutive_rejects rejected attempts in a row */
#define CATAPULT_ST_MAXSTEPS 3  /* max_steps attempts used */

typedef struct {
  int32_t coord;    /* CATAPULT_COORD_* */
  int32_t ncell[3]; /* interpolant cells per dimension, slowest -> fastest;
                       unique nodes per dimension = 3*ncell+1 */
  int32_t nfp;      /* field periods: the last grid dimension spans [lo, lo + 2pi/nfp) */
  int32_t nquant;   /* m, must equal CATAPULT_NQUANT_* of `coord` (Boozer: 4, or 1 = derivative-of-interpolant mode) */
  int32_t quant[16]; /* CATAPULT_Q_* tag of every column, or all zero (= the canonical order of `coord`) */
  double lo[3], hi[3]; /* Boozer: [0,1],[0,2pi],[0,2pi/nfp]; cyl: [Rmin,Rmax],[Zmin,Zmax],[0,2pi/nfp].
                          theta, zeta and phi are periodic with period hi-lo; s, R, Z extrapolate
                          with the nearest cell's cubic outside [lo,hi] */
  double G0, I0;       /* Boozer covariant components, constants (vacuum: I0 must be 0) */
  double iota0, iota1; /* rotational transform iota(s) = iota0 + iota1*s */
  double psi0;         /* Boozer: toroidal flux/(2pi) at s=1; cyl: psi_edge (loss level) */
  /* Non-vacuum Boozer ("vacuum, finite beta, etc."; R1b): 1-D profiles G(s), I(s), iota(s) on
     the unique s-nodes (iota "represented on a regular interpolant grid"): pointers to 3*ncell[0]+1
     doubles each -- device pointers for catapult_field_build, host pointers for catapult_field_build_host --
     all three or none.  NULL = vacuum: the scalars G0 (I0 = 0) and the linear law above.  The field keeps its
     own copy (the arrays may be freed after the call returns; for device arrays: after the stream has passed the
     call).  The profiles are interpolated by the tables' own piecewise cubic (value and derivative).  Every
     BASELINE config is vacuum; the shear Alfven wave is built on the vacuum model only. */
  const double *G_nodes, *I_nodes, *iota_nodes;
} catapult_field_desc;

typedef struct catapult_field catapult_field; /* opaque; owns the per-cell coefficient tables */

typedef struct {
  double mass, charge, energy; /* shared by all particles; v_total = sqrt(2E/m) */
  double T;                    /* end time of the trace (absolute time), > 0 and finite        */
  double rtol, atol;           /* Eq. 4; atol is multiplied by v_total for vpar
                                                                                   */
  double dt0, dtmax;           /* initial / maximum step; <= 0 selects the defaults of DESIGN.md S3 */
  int64_t max_steps;           /* attempts per particle PER CALL (every catapult_trace_continue
                                  window starts a new count); 0 = unlimited                     */
  int32_t max_consecutive_rejects; /* 0 = 500                                                   */
  int32_t saw_on;              /* 1: shear Alfven wave, Boozer only              */
  int32_t saw_m, saw_n;        /* Phi = Phi0 exp(-(s-s0)^2/w2) sin(m theta - n zeta + omega t)  */
  double saw_Phi0, saw_s0, saw_w2, saw_omega;
  int32_t loss_time_mode;      /* loss time tau: 0 = end time of the first accepted step that ends
                                  beyond the boundary, the end state returned (S5); 1 = root inside that
                                  step: cubic Hermite interpolant of the stepped variables through the step's end
                                  states and end derivatives, bisected to the first observed point beyond the
                                  boundary (Boozer: s >= 1; cylindrical: interpolated level function >= psi_edge,
                                  one table evaluation per bisection step), that point and its time
                                  returned (S5b)                                              */
  int32_t reserved_;           /* 0                                                              */
} catapult_trace_params;

/* ---- field tables ------------------------------------------------
 * catapult_field_build: d_nodes holds the unique nodes [nquant][3*ncell0+1][3*ncell1+1][3*ncell2+1]
 * (last index fastest).  A device kernel gathers, for every cell, the 4x4x4 nodal block of every
 * quantity (shared faces duplicated) and stores the cell's tricubic -- the SAME
 * polynomial as the Lagrange interpolant of those 64 nodes -- as its 64 coefficients
 * in the centred monomials w0^p0 w1^p1 w2^p2, w = 2u-1 (basis change in double-double arithmetic), in the
 * cell-major table [cell][quantity][64] (cell = (i0*ncell1+i1)*ncell2+i2; inside a 512-byte block the
 * coefficients are ordered by the power of theta (phi) first, then s (R), then zeta (Z): an internal
 * order).  One cell's coefficients of one quantity are four 128-byte lines.
 * catapult_field_export_rows recovers the nodal values in the paper's own row layout.  *out owns the
 * table (allocated stream-ordered on `stream`); d_nodes may be freed once the stream has run.
 * Errors: EINVAL (NULL, ncell<1 or more than 2^31-1 cells, nquant mismatch, hi<=lo, nfp<1, G0 == 0 for a
 * Boozer field -- also when profiles are given: G0 then only has to be non-zero, G(s) comes from G_nodes --,
 * only some of the three profile pointers), EUNSUPPORTED (a constant I0 != 0 without profiles: give I(s) as a
 * profile instead; non-canonical column order), ENOMEM, ECUDA.  When the build fails after the table was
 * allocated, the call waits for `stream` before it frees the table. */
catapult_status catapult_field_build(const catapult_field_desc *desc, const double *d_nodes,
                                     void *stream, catapult_field **out);
/* same with HOST nodes: copies them to the device, builds, synchronises, frees the staging copy */
catapult_status catapult_field_build_host(const catapult_field_desc *desc, const double *h_nodes,
                                          catapult_field **out);
catapult_status catapult_field_destroy(catapult_field *f);
/* bytes of the device coefficient table (64 * ncells * nquant * 8) */
size_t catapult_field_table_bytes(const catapult_field *f);

/* test hook: tricubic values of all quantities at npts points given in GRID coordinates
   d_pts[3][npts] ((s,theta,zeta) or (R,Z,phi), unreduced) -> d_out[nquant][npts] */
catapult_status catapult_field_eval(const catapult_field *f, int64_t npts, const double *d_pts,
                                    double *d_out, void *stream);
/* test hook: writes the table in the paper's own layout: row = cell*64 + node,
   column = quantity, d_out[(cell*64+node)*nquant + q]; 64*ncells*nquant doubles */
catapult_status catapult_field_export_rows(const catapult_field *f, double *d_out, void *stream);

/* ---- tracing --------------------------------------------------------------
 * catapult_trace: each of the n particles starts at t=0 from d_x0[4][n] and is advanced with
 * DP5 steps until min(tau, T): d_xf[4][n] = last observed state in the input's
 * coordinates (Boozer theta in (-pi,pi], zeta unreduced), d_tstop[n] = min(tau,T),
 * d_status[n] = CATAPULT_ST_*; d_nacc/d_nrej[n] (may be NULL) = accepted / rejected attempts.
 * A particle already outside at t=0 is returned unchanged with status LOST and t_stop = 0.
 * d_counters (may be NULL): CATAPULT_NCOUNTERS uint64 accumulated (atomically added) by the kernel:
 *   [0] accepted steps, [1] rejected attempts, [2] particles finished at T, [3] lost,
 *   [4] stalled, [5] max_steps, [6] right-hand-side evaluations, [7] cell fetches from the table,
 *   [8] of which blocking (the cell was not the one fetched ahead), [9] evaluation rounds of the
 *   32-slot blocks ([6] / (32 [9]) = fraction of slots doing useful work). */
#define CATAPULT_NCOUNTERS 10
catapult_status catapult_trace(const catapult_field *f, const catapult_trace_params *p, int64_t n,
                               const double *d_x0, double *d_xf, double *d_tstop,
                               int32_t *d_status, uint32_t *d_nacc, uint32_t *d_nrej,
                               uint64_t *d_counters, void *stream);
/* Restartable form: all arrays are in/out.  Particles whose d_status is REACHED_T are advanced
 * from their own time d_t[i] to p->T with controller step d_dt[i] and magnetic moment d_mu[i]
 * (per unit mass); others are left untouched.  d_nacc/d_nrej (may be NULL) are incremented.
 * catapult_trace_init fills (t=0, dt=dt0, mu from the tabulated |B|, status REACHED_T or LOST)
 * so that init + continue(T) equals catapult_trace(T) exactly. */
catapult_status catapult_trace_init(const catapult_field *f, const catapult_trace_params *p,
                                    int64_t n, const double *d_x, double *d_t, double *d_dt,
                                    double *d_mu, int32_t *d_status, void *stream);
catapult_status catapult_trace_continue(const catapult_field *f, const catapult_trace_params *p,
                                        int64_t n, double *d_x, double *d_t, double *d_dt,
                                        double *d_mu, int32_t *d_status, uint32_t *d_nacc,
                                        uint32_t *d_nrej, uint64_t *d_counters, void *stream);
/* HOST-buffer form of catapult_trace: copies h_x0 to the device, traces, copies the results back
   and synchronises.  h_nacc/h_nrej/h_counters may be NULL.  The *_host calls keep one device staging
   slab and one non-blocking stream per host thread between calls (grown on demand);
   catapult_release_host_cache frees the calling thread's.  Nothing frees them at thread exit (the CUDA
   context may already be gone by then): a thread that used a *_host call and ends without calling
   catapult_release_host_cache leaves its slab and stream allocated until the process ends.  Pinned host
   buffers make the copies asynchronous with respect to the host. */
catapult_status catapult_trace_host(const catapult_field *f, const catapult_trace_params *p,
                                    int64_t n, const double *h_x0, double *h_xf, double *h_tstop,
                                    int32_t *h_status, uint32_t *h_nacc, uint32_t *h_nrej,
                                    uint64_t *h_counters);
/* HOST-buffer form of catapult_trace_continue: the state arrays (all required except h_nacc,
   h_nrej, h_counters) are copied to the device, advanced to p->T, copied back; synchronises. */
catapult_status catapult_trace_continue_host(const catapult_field *f, const catapult_trace_params *p,
                                             int64_t n, double *h_x, double *h_t, double *h_dt,
                                             double *h_mu, int32_t *h_status, uint32_t *h_nacc,
                                             uint32_t *h_nrej, uint64_t *h_counters);
catapult_status catapult_release_host_cache(void);
/* test hook: scripted replay.  Every particle starts at t = 0 from d_x0[4][n] and takes the step sizes
   d_h[nsteps][n] (step-major) one after the other, each step ACCEPTED whatever its error ratio (the
   controller is bypassed); a particle stops at its first h <= 0, after nsteps steps, or when an end
   state is beyond the loss boundary.  d_r[nsteps][n] (may be NULL) receives Eq. 4's error ratio of every
   step taken (other entries are left untouched).  d_xf, d_tstop, d_status as in catapult_trace
   (status REACHED_T when the script ran out).  Adaptive runs in different arithmetic take different
   accept/reject decisions and then differ by their global error; replaying one
   run's accepted step sizes removes the decisions and leaves the step arithmetic to be compared. */
catapult_status catapult_trace_scripted(const catapult_field *f, const catapult_trace_params *p, int64_t n,
                                        const double *d_x0, int32_t nsteps, const double *d_h,
                                        double *d_xf, double *d_tstop, int32_t *d_status, double *d_r,
                                        void *stream);
/* test hook: ONE attempted DP5 step of size d_h[i] from state d_x[4][n] at time d_t[n] (mu taken
   from the state as in catapult_trace_init): d_xnew[4][n], d_errratio[n] (Eq. 4),
   d_k[7][4][n] = the seven stage derivatives in the stepped variables */
catapult_status catapult_step_once(const catapult_field *f, const catapult_trace_params *p,
                                   int64_t n, const double *d_x, const double *d_t,
                                   const double *d_h, double *d_xnew, double *d_errratio,
                                   double *d_k, void *stream);

/* ---- estimate (Eq. 2) ----------------------------------------------------------
 * g_kind 0: g = 1[status == LOST] (integer count, exact); 1: g = t_stop; 2: g = d_g_user.
 * d_out[4] (device, required) = { mean, standard error sqrt((sum g^2/n - mean^2)/(n-1)), sum g, sum g^2 }:
 * the two sums (with n) are what a particle-sharded run reduces over its ranks (24 bytes).
 * Deterministic fixed-order tree.  If h_out != NULL the four doubles are also copied to the host
 * and the stream is synchronised. */
catapult_status catapult_estimate(int32_t g_kind, int64_t n, const int32_t *d_status,
                                  const double *d_tstop, const double *d_g_user, double *d_out,
                                  double *h_out, void *stream);

/* ---- other measurements g on the end states ("Similar functions g can be chosen to calculate energy
 * loss ..., wall-loads from alpha particles"; readings G2, G3) ---------------------------------------
 * catapult_measure_lost_energy: d_g[i] = 1[status LOST] * (vpar^2/2 + mu_i |B|(x_f,i)) / (v_total^2/2): the energy a
 * lost particle leaves with, in units of the birth energy all particles share, |B| from the field's
 * tables at the exit point d_xf[4][n] (as returned by the tracing calls), d_mu[n] the magnetic moment per unit mass
 * (catapult_trace_init / catapult_trace_continue keep it).  Feed d_g to catapult_estimate with g_kind 2: the mean is
 * the fraction of the alpha power lost (equal to the loss fraction in a static field, not with a wave).
 * Errors: EINVAL (NULL, n < 0, bad params as in catapult_trace, another device), ECUDA. */
catapult_status catapult_measure_lost_energy(const catapult_field *f, const catapult_trace_params *p, int64_t n,
                                             const double *d_xf, const double *d_mu, const int32_t *d_status,
                                             double *d_g, void *stream);
/* catapult_exit_histogram: the wall-load stand-in.  d_hist[nbins0][nbins1] (uint64, zeroed by the call) = number of
 * LOST particles per bin of the exit point: Boozer (theta over [0, 2pi), zeta over one field period), both periodic;
 * cylindrical (phi = atan2(y, x) over one field period, periodic; Z over the grid's [lo, hi], end bins collect what
 * lies outside).  Bin of a coordinate a: u = (a - lo) / (hi - lo), minus floor(u) when periodic, floor(u * nbins)
 * clamped to [0, nbins-1], each operation rounded once.  Exact integer counts whatever the launch order.
 * Errors: EINVAL (NULL, n < 0, nbins < 1 or more than 2^24 bins, another device), ECUDA. */
catapult_status catapult_exit_histogram(const catapult_field *f, int64_t n, const double *d_xf,
                                        const int32_t *d_status, int32_t nbins0, int32_t nbins1, uint64_t *d_hist,
                                        void *stream);

/* ---- the estimate for callers that must not allocate device memory ------------------------------
 * catapult_estimate above takes a few KiB of device scratch from the stream-ordered allocator on every call.
 * Some programs cannot have a library do that on their behalf: a service that hands the whole GPU to its own
 * memory manager at start-up and treats any later driver allocation as a bug (or simply has nothing left to
 * give); a control loop with a latency budget, where an allocation may stall on the driver's lock or fail at
 * the worst moment; a driver set-up without memory-pool support, where cudaMallocAsync is not available at
 * all.  For them catapult_estimate_static computes the same four numbers -- same block partition, same
 * summation order, so bit-identical to catapult_estimate -- and calls no cudaMalloc / cudaFree /
 * cudaMallocAsync or any other allocating routine.  The caller passes the inputs and d_out[4] exactly as for
 * catapult_estimate (g_kind, NULL rules and errors are the same; there is no host copy: read d_out yourself).
 *
 * Where the scratch lives: in a 16 KiB array that is part of libcatapult.so's device image (one pair of
 * partial sums per block of 2048 particles).  Every GPU that loads the library carries these 16 KiB until the
 * process exits, whether or not this function is ever called.
 * Limit: n <= CATAPULT_ESTIMATE_STATIC_MAX_N (2,097,152 particles = 1024 blocks; twice BASELINE's largest
 * ensemble).  A larger n is refused with CATAPULT_EINVAL and a message that names the limit; nothing is launched.
 * First call on a device: looks up the array's address on that device (once; the current device must be the
 * one `stream` belongs to, as for every call of this library).  Make that first call during set-up, before any
 * stream capture is begun.
 * Sharing: all calls on one GPU use the same array.  Calls on one stream follow each other and are safe.  Two
 * calls that can run at the same time on one GPU (different streams, different host threads) overwrite each
 * other's partial sums and return garbage without any error: serialise them yourself (one stream, or an event
 * between them).  The array keeps the last call's partial sums; no call depends on them, every slot that is
 * read has been written by the same call first. */
#define CATAPULT_ESTIMATE_STATIC_MAX_N 2097152LL
catapult_status catapult_estimate_static(int32_t g_kind, int64_t n, const int32_t *d_status,
                                         const double *d_tstop, const double *d_g_user, double *d_out,
                                         void *stream);

/* launch geometry the tracer uses on the current device: persistent blocks and threads per block */
catapult_status catapult_trace_launch_shape(const catapult_field *f, const catapult_trace_params *p,
                                            int32_t *blocks, int32_t *threads);

const char *catapult_last_error(void);
const char *catapult_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CATAPULT_H */
