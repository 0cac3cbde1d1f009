// C-ABI entry points of libcatapult.so (include/catapult.h): argument validation, table ownership,
// parameter packing and stream-ordered launches.  No arithmetic of the method lives here.
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "gc_device.cuh"

namespace catapult {

static thread_local std::string g_last_error;

void set_error(const std::string& msg) { g_last_error = msg; }

catapult_status cuda_fail(cudaError_t e, const char* what) {
  char buf[512];
  std::snprintf(buf, sizeof(buf), "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
  set_error(buf);
  return e == cudaErrorMemoryAllocation ? CATAPULT_ENOMEM : CATAPULT_ECUDA;
}

static catapult_status fail(catapult_status st, const char* msg) {
  set_error(msg);
  return st;
}

static const double PI = 3.14159265358979323846;

static catapult_status validate_desc(const catapult_field_desc* d) {
  if (!d) return fail(CATAPULT_EINVAL, "desc is NULL");
  if (d->coord != CATAPULT_COORD_BOOZER && d->coord != CATAPULT_COORD_CYL)
    return fail(CATAPULT_EINVAL, "desc.coord must be CATAPULT_COORD_BOOZER or CATAPULT_COORD_CYL");
  long long ncells = 1;
  for (int i = 0; i < 3; ++i) {
    if (d->ncell[i] < 1) return fail(CATAPULT_EINVAL, "desc.ncell must be >= 1");
    if (!(std::isfinite(d->lo[i]) && std::isfinite(d->hi[i]) && d->hi[i] > d->lo[i]))
      return fail(CATAPULT_EINVAL, "desc.lo/hi must be finite with hi > lo");
    // the kernels carry a flat cell index in 32 bits and node indices 3*ncell+1 per dimension
    if (d->ncell[i] > (INT32_MAX - 1) / 3) return fail(CATAPULT_EINVAL, "desc.ncell is too large");
    ncells *= d->ncell[i];
    if (ncells > (long long)INT32_MAX) return fail(CATAPULT_EINVAL, "desc.ncell: more than 2^31-1 cells");
  }
  // Boozer with ONE quantity: the derivative-of-interpolant mode (only |B| tabulated, R1c)
  const bool doi = d->coord == CATAPULT_COORD_BOOZER && d->nquant == CATAPULT_NQUANT_BOOZER_DOI;
  const int want = doi ? CATAPULT_NQUANT_BOOZER_DOI
                       : (d->coord == CATAPULT_COORD_BOOZER ? CATAPULT_NQUANT_BOOZER : CATAPULT_NQUANT_CYL);
  if (d->nquant != want)
    return fail(CATAPULT_EINVAL, "desc.nquant does not match desc.coord (Boozer: 4, or 1 = derivative-of-interpolant mode; cyl: 7)");
  // semantic tags of the columns: all zero = the canonical order of `coord`; anything else must spell it out
  bool tagged = false;
  for (int i = 0; i < 16; ++i) tagged = tagged || d->quant[i] != 0;
  if (tagged) {
    static const int32_t BZ[4] = {CATAPULT_Q_MODB, CATAPULT_Q_DMODB_DS, CATAPULT_Q_DMODB_DTHETA, CATAPULT_Q_DMODB_DZETA};
    static const int32_t CY[7] = {CATAPULT_Q_B_R,        CATAPULT_Q_B_PHI,    CATAPULT_Q_B_Z,      CATAPULT_Q_DMODB_DR,
                                  CATAPULT_Q_DMODB_DPHI_OVER_R, CATAPULT_Q_DMODB_DZ, CATAPULT_Q_PSI_LEVEL};
    const int32_t* canon = d->coord == CATAPULT_COORD_BOOZER ? BZ : CY;
    for (int i = 0; i < 16; ++i)
      if (d->quant[i] != (i < want ? canon[i] : 0))
        return fail(CATAPULT_EUNSUPPORTED, "desc.quant: only the canonical column order of `coord` is built");
  }
  if (d->nfp < 1) return fail(CATAPULT_EINVAL, "desc.nfp must be >= 1");
  if (d->coord == CATAPULT_COORD_BOOZER) {
    const int nprof = (d->G_nodes != nullptr) + (d->I_nodes != nullptr) + (d->iota_nodes != nullptr);
    if (nprof != 0 && nprof != 3)
      return fail(CATAPULT_EINVAL, "G_nodes, I_nodes and iota_nodes: give all three (non-vacuum Boozer) or none");
    if (nprof == 0 && d->I0 != 0.0)
      return fail(CATAPULT_EUNSUPPORTED, "non-vacuum Boozer is built with tabulated profiles: give G_nodes, I_nodes, iota_nodes");
    if (!(std::isfinite(d->G0) && d->G0 != 0.0)) return fail(CATAPULT_EINVAL, "desc.G0 must be finite, non-zero");
    if (!(std::isfinite(d->psi0) && d->psi0 != 0.0)) return fail(CATAPULT_EINVAL, "desc.psi0 must be finite, non-zero");
  } else {
    if (d->G_nodes || d->I_nodes || d->iota_nodes)
      return fail(CATAPULT_EINVAL, "profiles on the s-nodes belong to Boozer tracing");
    if (!std::isfinite(d->psi0)) return fail(CATAPULT_EINVAL, "desc.psi0 (psi_edge) must be finite");
  }
  return CATAPULT_OK;
}

static void fill_field_const(const catapult_field_desc& d, const double* table, const double* node0,
                             FieldConst* fc) {
  fc->table = table;
  fc->node0 = node0;
  fc->prof = d.G_nodes ? node0 + 1 : nullptr;  // the field's own copy of the three profiles sits behind node0
  fc->coord = d.coord;
  fc->m = d.nquant;
  for (int i = 0; i < 3; ++i) {
    fc->k[i] = d.ncell[i];
    fc->lo[i] = d.lo[i];
    fc->span[i] = d.hi[i] - d.lo[i];
    fc->invspan[i] = 1.0 / fc->span[i];
    const double h = fc->span[i] / (double)d.ncell[i];
    fc->invh[i] = 1.0 / h;
  }
  fc->G = d.G0;
  fc->invG = d.G0 != 0.0 ? 1.0 / d.G0 : 0.0;
  fc->psi0 = d.psi0;
  fc->invpsi0 = d.psi0 != 0.0 ? 1.0 / d.psi0 : 0.0;
  fc->iota0 = d.iota0;
  fc->iota1 = d.iota1;
}

static catapult_status make_trace_const(const catapult_field* f, const catapult_trace_params* p, TraceConst* tc,
                                        int* model) {
  if (!f) return fail(CATAPULT_EINVAL, "field is NULL");
  if (!p) return fail(CATAPULT_EINVAL, "params is NULL");
  if (!(std::isfinite(p->mass) && p->mass > 0.0 && std::isfinite(p->charge) && p->charge != 0.0 &&
        std::isfinite(p->energy) && p->energy > 0.0))
    return fail(CATAPULT_EINVAL, "mass, |charge| and energy must be finite and positive");
  if (!(std::isfinite(p->T) && p->T > 0.0)) return fail(CATAPULT_EINVAL, "T must be finite and > 0");
  if (!(std::isfinite(p->rtol) && p->rtol >= 0.0 && std::isfinite(p->atol) && p->atol >= 0.0 &&
        (p->rtol > 0.0 || p->atol > 0.0)))
    return fail(CATAPULT_EINVAL, "rtol/atol must be finite, non-negative, not both zero");
  if (p->max_steps < 0 || p->max_consecutive_rejects < 0)
    return fail(CATAPULT_EINVAL, "max_steps / max_consecutive_rejects must be >= 0");
  if (p->loss_time_mode != 0 && p->loss_time_mode != 1) return fail(CATAPULT_EINVAL, "loss_time_mode must be 0 or 1");
  if (p->saw_on) {
    if (f->desc.coord != CATAPULT_COORD_BOOZER)
      return fail(CATAPULT_EUNSUPPORTED, "the shear Alfven wave is built for Boozer tracing only");
    if (!(std::isfinite(p->saw_omega) && p->saw_omega != 0.0 && std::isfinite(p->saw_w2) && p->saw_w2 > 0.0 &&
          std::isfinite(p->saw_Phi0) && std::isfinite(p->saw_s0)))
      return fail(CATAPULT_EINVAL, "saw_omega must be non-zero, saw_w2 > 0, saw_Phi0/saw_s0 finite");
  }
  tc->f = f->fc;
  tc->M = p->mass;
  tc->invM = 1.0 / p->mass;
  tc->q = p->charge;
  tc->Moq = p->mass / p->charge;
  tc->vtot = std::sqrt(2.0 * p->energy / p->mass);
  tc->vtot2 = tc->vtot * tc->vtot;
  tc->T = p->T;
  tc->rtol = p->rtol;
  tc->atol = p->atol;
  // DESIGN.md S3 defaults: dtmax = (pi/2) L / v_total, dt0 = 1e-3 dtmax.  Boozer: L = |G| / |B|(node 0); the
  // node value is on the device (field_build_kernel leaves it next to the table), so dtmax <= 0 is passed on
  // and the tracer kernel resolves both defaults itself -- no host read-back, no synchronisation.
  double dtmax = p->dtmax, dt0 = p->dt0;
  if (!(dtmax > 0.0)) {
    if (f->desc.coord == CATAPULT_COORD_CYL) dtmax = 0.5 * PI * f->desc.hi[0] / tc->vtot;  // L = R_max
    else dtmax = 0.0;
  }
  if (dtmax > 0.0) {
    dt0 = dt0 > 0.0 ? dt0 : 1e-3 * dtmax;
    if (dt0 > dtmax) dt0 = dtmax;
  }
  tc->dt0 = dt0;
  tc->dtmax = dtmax;
  tc->max_steps = p->max_steps;
  tc->max_rej = p->max_consecutive_rejects > 0 ? p->max_consecutive_rejects : 500;
  tc->loss_time_mode = p->loss_time_mode;
  tc->saw_m = p->saw_m;
  tc->saw_n = p->saw_n;
  tc->saw_Phi0 = p->saw_Phi0;
  tc->saw_s0 = p->saw_s0;
  tc->saw_invw2 = p->saw_on ? 1.0 / p->saw_w2 : 0.0;
  tc->saw_omega = p->saw_omega;
  tc->saw_inv_omG = p->saw_on ? f->fc.invG / p->saw_omega : 0.0;
  if (f->fc.prof && p->saw_on)
    return fail(CATAPULT_EUNSUPPORTED, "the shear Alfven wave is built on the vacuum Boozer model only");
  *model = f->desc.coord == CATAPULT_COORD_CYL
               ? MODEL_CART
               : (f->fc.prof ? MODEL_BOOZER_NV : (p->saw_on ? MODEL_BOOZER_SAW : MODEL_BOOZER_VAC));
  return CATAPULT_OK;
}

// Every call that reads the tables on `s` is ordered after the build, whatever stream the build ran on.
static catapult_status use_field_on(const catapult_field* f, cudaStream_t s) {
  int dev = -1;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  if (dev != f->device) return fail(CATAPULT_EINVAL, "field was built on another device than the current one");
  CATAPULT_CUDA_TRY(cudaStreamWaitEvent(s, f->built, 0));
  return CATAPULT_OK;
}
static catapult_status use_device_of(const catapult_field* f) {
  int dev = -1;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  if (dev != f->device) return fail(CATAPULT_EINVAL, "field was built on another device than the current one");
  return CATAPULT_OK;
}

}  // namespace catapult

using namespace catapult;

extern "C" {

const char* catapult_last_error(void) { return g_last_error.c_str(); }
const char* catapult_version(void) { return "catapult-b200 0.1 (sm_100a)"; }

catapult_status catapult_field_build(const catapult_field_desc* desc, const double* d_nodes, void* stream,
                                     catapult_field** out) {
  catapult_status st = validate_desc(desc);
  if (st != CATAPULT_OK) return st;
  if (!d_nodes) return fail(CATAPULT_EINVAL, "d_nodes is NULL");
  if (!out) return fail(CATAPULT_EINVAL, "out is NULL");
  *out = nullptr;
  catapult_field* f = new (std::nothrow) catapult_field();
  if (!f) return fail(CATAPULT_ENOMEM, "host allocation failed");
  f->desc = *desc;
  f->ncells = (int64_t)desc->ncell[0] * desc->ncell[1] * desc->ncell[2];
  f->table_bytes = (size_t)f->ncells * desc->nquant * 64 * sizeof(double);
  f->d_table = nullptr;
  f->built = nullptr;
  // stream-ordered allocation: the build neither blocks the host nor synchronises the device
  cudaError_t e = cudaGetDevice(&f->device);
  const size_t nprof = desc->G_nodes ? (size_t)(3 * desc->ncell[0] + 1) : 0;  // non-vacuum Boozer: three profiles
  if (e == cudaSuccess)
    e = cudaMallocAsync((void**)&f->d_table, f->table_bytes + (1 + 3 * nprof) * sizeof(double), (cudaStream_t)stream);
  if (e != cudaSuccess) {
    delete f;
    return cuda_fail(e, "cudaMallocAsync(table)");
  }
  double* d_node0 = f->d_table + f->table_bytes / sizeof(double);
  fill_field_const(*desc, f->d_table, d_node0, &f->fc);
  st = launch_field_build(*desc, d_nodes, f->d_table, d_node0, (cudaStream_t)stream);
  if (st == CATAPULT_OK && nprof) {  // the field keeps its own copy: the caller's arrays may go after this call
    const double* src[3] = {desc->G_nodes, desc->I_nodes, desc->iota_nodes};
    for (int k = 0; k < 3 && e == cudaSuccess; ++k)
      e = cudaMemcpyAsync(d_node0 + 1 + k * nprof, src[k], nprof * sizeof(double), cudaMemcpyDefault,
                          (cudaStream_t)stream);
    if (e != cudaSuccess) st = cuda_fail(e, "cudaMemcpyAsync(profiles)");
    f->desc.G_nodes = f->desc.I_nodes = f->desc.iota_nodes = d_node0 + 1;  // marks "non-vacuum"; not the caller's
  }
  if (st == CATAPULT_OK) {
    e = cudaEventCreateWithFlags(&f->built, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventRecord(f->built, (cudaStream_t)stream);
    if (e != cudaSuccess) st = cuda_fail(e, "cudaEventRecord(built)");
  }
  if (st != CATAPULT_OK) {
    // the table came from cudaMallocAsync: cudaFree does not wait for work that still uses it, and the build kernel or
    // the profile copies may be in flight on `stream`
    cudaStreamSynchronize((cudaStream_t)stream);
    if (f->built) cudaEventDestroy(f->built);
    cudaFree(f->d_table);
    delete f;
    return st;
  }
  *out = f;
  return CATAPULT_OK;
}

catapult_status catapult_field_build_host(const catapult_field_desc* desc, const double* h_nodes,
                                          catapult_field** out) {
  catapult_status st = validate_desc(desc);
  if (st != CATAPULT_OK) return st;
  if (!h_nodes) return fail(CATAPULT_EINVAL, "h_nodes is NULL");
  if (!out) return fail(CATAPULT_EINVAL, "out is NULL");
  size_t nn = (size_t)desc->nquant;
  for (int i = 0; i < 3; ++i) nn *= (size_t)(3 * desc->ncell[i] + 1);
  double* d_nodes = nullptr;
  CATAPULT_CUDA_TRY(cudaMalloc((void**)&d_nodes, nn * sizeof(double)));
  cudaError_t e = cudaMemcpy(d_nodes, h_nodes, nn * sizeof(double), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(d_nodes);
    return cuda_fail(e, "cudaMemcpy(nodes)");
  }
  st = catapult_field_build(desc, d_nodes, nullptr, out);
  e = cudaDeviceSynchronize();
  cudaFree(d_nodes);
  if (st == CATAPULT_OK && e != cudaSuccess) {
    catapult_field_destroy(*out);
    *out = nullptr;
    return cuda_fail(e, "field build");
  }
  return st;
}

catapult_status catapult_field_destroy(catapult_field* f) {
  if (!f) return CATAPULT_OK;
  // The table is a stream-ordered allocation, and for those cudaFree returns the memory WITHOUT waiting for kernels
  // that still read it (unlike memory from cudaMalloc).  Traces and evaluations of this field may be running on any
  // stream of its device, so the whole device is drained first; otherwise `del field` right after an asynchronous
  // trace would hand the table to the next allocation under the running tracer.
  int cur = -1;
  cudaError_t e = cudaGetDevice(&cur);
  if (e == cudaSuccess && cur != f->device) e = cudaSetDevice(f->device);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  if (f->built) cudaEventDestroy(f->built);
  if (f->d_table) cudaFree(f->d_table);
  if (cur >= 0 && cur != f->device) cudaSetDevice(cur);
  delete f;
  // an error left behind by earlier asynchronous work is reported, but the field is gone either way
  if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceSynchronize before freeing the field's table");
  return CATAPULT_OK;
}

size_t catapult_field_table_bytes(const catapult_field* f) { return f ? f->table_bytes : 0; }

catapult_status catapult_field_eval(const catapult_field* f, int64_t npts, const double* d_pts, double* d_out,
                                    void* stream) {
  if (!f) return fail(CATAPULT_EINVAL, "field is NULL");
  if (npts < 0) return fail(CATAPULT_EINVAL, "npts < 0");
  if (npts > 0 && (!d_pts || !d_out)) return fail(CATAPULT_EINVAL, "d_pts/d_out is NULL");
  catapult_status st = use_field_on(f, (cudaStream_t)stream);
  if (st != CATAPULT_OK) return st;
  return launch_field_eval(f->fc, npts, d_pts, d_out, (cudaStream_t)stream);
}

catapult_status catapult_field_export_rows(const catapult_field* f, double* d_out, void* stream) {
  if (!f || !d_out) return fail(CATAPULT_EINVAL, "field/d_out is NULL");
  catapult_status st = use_field_on(f, (cudaStream_t)stream);
  if (st != CATAPULT_OK) return st;
  return launch_field_export_rows(f->fc, f->ncells, d_out, (cudaStream_t)stream);
}

static catapult_status run_trace(const catapult_field* f, const catapult_trace_params* p, TraceArgs a,
                                 cudaStream_t s, bool scripted = false) {
  TraceConst tc;
  int model = 0;
  catapult_status st = make_trace_const(f, p, &tc, &model);
  if (st != CATAPULT_OK) return st;
  st = use_field_on(f, s);
  if (st != CATAPULT_OK) return st;
  if (a.n == 0) return CATAPULT_OK;
  unsigned long long* queue = nullptr;
  CATAPULT_CUDA_TRY(cudaMallocAsync((void**)&queue, TRACE_SCRATCH_BYTES, s));
  cudaError_t e = cudaMemsetAsync(queue, 0, TRACE_SCRATCH_BYTES, s);
  if (e != cudaSuccess) {
    cudaFreeAsync(queue, s);
    return cuda_fail(e, "cudaMemsetAsync(queue)");
  }
  a.queue = queue;
  st = launch_trace(tc, a, model, scripted ? 1 : 0, s);
  cudaFreeAsync(queue, s);
  return st;
}

catapult_status catapult_trace(const catapult_field* f, const catapult_trace_params* p, int64_t n, const double* d_x0,
                               double* d_xf, double* d_tstop, int32_t* d_status, uint32_t* d_nacc, uint32_t* d_nrej,
                               uint64_t* d_counters, void* stream) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (n > 0 && (!d_x0 || !d_xf || !d_tstop || !d_status))
    return fail(CATAPULT_EINVAL, "d_x0, d_xf, d_tstop and d_status are required");
  TraceArgs a{};
  a.n = n;
  a.x_in = d_x0;
  a.x_out = d_xf;
  a.t_io = d_tstop;
  a.status = d_status;
  a.nacc = d_nacc;
  a.nrej = d_nrej;
  a.counters = (unsigned long long*)d_counters;
  return run_trace(f, p, a, (cudaStream_t)stream);
}

catapult_status catapult_trace_scripted(const catapult_field* f, const catapult_trace_params* p, int64_t n,
                                        const double* d_x0, int32_t nsteps, const double* d_h, double* d_xf,
                                        double* d_tstop, int32_t* d_status, double* d_r, void* stream) {
  if (n < 0 || nsteps < 0) return fail(CATAPULT_EINVAL, "n < 0 or nsteps < 0");
  if (n > 0 && (!d_x0 || !d_xf || !d_tstop || !d_status || (nsteps > 0 && !d_h)))
    return fail(CATAPULT_EINVAL, "d_x0, d_h, d_xf, d_tstop and d_status are required");
  TraceArgs a{};
  a.n = n;
  a.x_in = d_x0;
  a.x_out = d_xf;
  a.t_io = d_tstop;
  a.status = d_status;
  a.script_h = d_h;
  a.script_r = d_r;
  a.script_len = nsteps;
  return run_trace(f, p, a, (cudaStream_t)stream, true);
}

catapult_status catapult_trace_init(const catapult_field* f, const catapult_trace_params* p, int64_t n,
                                    const double* d_x, double* d_t, double* d_dt, double* d_mu, int32_t* d_status,
                                    void* stream) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (n > 0 && (!d_x || !d_t || !d_dt || !d_mu || !d_status))
    return fail(CATAPULT_EINVAL, "d_x, d_t, d_dt, d_mu and d_status are required");
  TraceArgs a{};
  a.n = n;
  a.x_in = d_x;
  a.x_out = const_cast<double*>(d_x);  // only rewritten (unchanged) for particles born outside
  a.t_io = d_t;
  a.dt_io = d_dt;
  a.mu_io = d_mu;
  a.status = d_status;
  a.init_only = 1;
  return run_trace(f, p, a, (cudaStream_t)stream);
}

catapult_status catapult_trace_continue(const catapult_field* f, const catapult_trace_params* p, int64_t n,
                                        double* d_x, double* d_t, double* d_dt, double* d_mu, int32_t* d_status,
                                        uint32_t* d_nacc, uint32_t* d_nrej, uint64_t* d_counters, void* stream) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (n > 0 && (!d_x || !d_t || !d_dt || !d_mu || !d_status))
    return fail(CATAPULT_EINVAL, "d_x, d_t, d_dt, d_mu and d_status are required");
  TraceArgs a{};
  a.n = n;
  a.x_in = d_x;
  a.x_out = d_x;
  a.t_io = d_t;
  a.dt_io = d_dt;
  a.mu_io = d_mu;
  a.status = d_status;
  a.nacc = d_nacc;
  a.nrej = d_nrej;
  a.counters = (unsigned long long*)d_counters;
  a.resume = 1;
  return run_trace(f, p, a, (cudaStream_t)stream);
}

// ---- HOST-buffer forms -------------------------------------------------------------------------------------
// One staging slab and one non-blocking stream per host thread, kept between calls (grown on demand, released
// by catapult_release_host_cache): the copies and the kernel are enqueued back to back on that stream and the
// call returns after one cudaStreamSynchronize.
namespace {
struct HostCache {
  int device = -1;
  cudaStream_t stream = nullptr;
  char* slab = nullptr;
  size_t bytes = 0;
  void release() {
    if (slab) cudaFree(slab);
    if (stream) cudaStreamDestroy(stream);
    slab = nullptr;
    stream = nullptr;
    bytes = 0;
    device = -1;
  }
  ~HostCache() {}  // at thread exit the CUDA context may be gone already: nothing is freed here
};
thread_local HostCache g_host;

catapult_status host_slab(const catapult_field* f, size_t bytes, char** slab, cudaStream_t* stream) {
  catapult_status st = use_device_of(f);
  if (st != CATAPULT_OK) return st;
  if (g_host.device != f->device) g_host.release();
  if (!g_host.stream) {
    CATAPULT_CUDA_TRY(cudaStreamCreateWithFlags(&g_host.stream, cudaStreamNonBlocking));
    g_host.device = f->device;
  }
  if (g_host.bytes < bytes) {
    if (g_host.slab) cudaFree(g_host.slab);
    g_host.slab = nullptr;
    g_host.bytes = 0;
    CATAPULT_CUDA_TRY(cudaMalloc((void**)&g_host.slab, bytes));
    g_host.bytes = bytes;
  }
  *slab = g_host.slab;
  *stream = g_host.stream;
  return CATAPULT_OK;
}
}  // namespace

catapult_status catapult_release_host_cache(void) {
  g_host.release();
  return CATAPULT_OK;
}

catapult_status catapult_trace_host(const catapult_field* f, const catapult_trace_params* p, int64_t n,
                                    const double* h_x0, double* h_xf, double* h_tstop, int32_t* h_status,
                                    uint32_t* h_nacc, uint32_t* h_nrej, uint64_t* h_counters) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (n > 0 && (!h_x0 || !h_xf || !h_tstop || !h_status))
    return fail(CATAPULT_EINVAL, "h_x0, h_xf, h_tstop and h_status are required");
  if (!f || !p) return fail(CATAPULT_EINVAL, "field/params is NULL");
  if (n == 0) return CATAPULT_OK;
  // one device slab: x0[4n] xf[4n] tstop[n] | counters | status[n] nacc[n] nrej[n]
  const size_t nd = (size_t)n;
  const size_t bytes = nd * 9 * sizeof(double) + CATAPULT_NCOUNTERS * sizeof(uint64_t) + nd * 3 * sizeof(uint32_t) + 64;
  char* slab = nullptr;
  cudaStream_t s = nullptr;
  catapult_status st = host_slab(f, bytes, &slab, &s);
  if (st != CATAPULT_OK) return st;
  double* d_x0 = (double*)slab;
  double* d_xf = d_x0 + 4 * nd;
  double* d_ts = d_xf + 4 * nd;
  uint64_t* d_cnt = (uint64_t*)(d_ts + nd);
  int32_t* d_st = (int32_t*)(d_cnt + CATAPULT_NCOUNTERS);
  uint32_t* d_na = (uint32_t*)(d_st + nd);
  uint32_t* d_nr = d_na + nd;
  const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
  cudaError_t e = cudaMemcpyAsync(d_x0, h_x0, 4 * nd * sizeof(double), H2D, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_cnt, 0, CATAPULT_NCOUNTERS * sizeof(uint64_t), s);
  if (e == cudaSuccess) {
    st = catapult_trace(f, p, n, d_x0, d_xf, d_ts, d_st, d_na, d_nr, d_cnt, s);
    if (st == CATAPULT_OK) {
      e = cudaMemcpyAsync(h_xf, d_xf, 4 * nd * sizeof(double), D2H, s);
      if (e == cudaSuccess) e = cudaMemcpyAsync(h_tstop, d_ts, nd * sizeof(double), D2H, s);
      if (e == cudaSuccess) e = cudaMemcpyAsync(h_status, d_st, nd * sizeof(int32_t), D2H, s);
      if (e == cudaSuccess && h_nacc) e = cudaMemcpyAsync(h_nacc, d_na, nd * sizeof(uint32_t), D2H, s);
      if (e == cudaSuccess && h_nrej) e = cudaMemcpyAsync(h_nrej, d_nr, nd * sizeof(uint32_t), D2H, s);
      if (e == cudaSuccess && h_counters)
        e = cudaMemcpyAsync(h_counters, d_cnt, CATAPULT_NCOUNTERS * sizeof(uint64_t), D2H, s);
    }
  }
  cudaError_t e2 = cudaStreamSynchronize(s);
  if (st != CATAPULT_OK) return st;
  if (e != cudaSuccess) return cuda_fail(e, "catapult_trace_host copies");
  if (e2 != cudaSuccess) return cuda_fail(e2, "catapult_trace_host");
  return CATAPULT_OK;
}

catapult_status catapult_trace_continue_host(const catapult_field* f, const catapult_trace_params* p, int64_t n,
                                             double* h_x, double* h_t, double* h_dt, double* h_mu, int32_t* h_status,
                                             uint32_t* h_nacc, uint32_t* h_nrej, uint64_t* h_counters) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (n > 0 && (!h_x || !h_t || !h_dt || !h_mu || !h_status))
    return fail(CATAPULT_EINVAL, "h_x, h_t, h_dt, h_mu and h_status are required");
  if (!f || !p) return fail(CATAPULT_EINVAL, "field/params is NULL");
  if (n == 0) return CATAPULT_OK;
  // one device slab: x[4n] t[n] dt[n] mu[n] | counters | status[n] nacc[n] nrej[n]
  const size_t nd = (size_t)n;
  const size_t bytes = nd * 7 * sizeof(double) + CATAPULT_NCOUNTERS * sizeof(uint64_t) + nd * 3 * sizeof(uint32_t) + 64;
  char* slab = nullptr;
  cudaStream_t s = nullptr;
  catapult_status st = host_slab(f, bytes, &slab, &s);
  if (st != CATAPULT_OK) return st;
  double* d_x = (double*)slab;
  double* d_t = d_x + 4 * nd;
  double* d_dt = d_t + nd;
  double* d_mu = d_dt + nd;
  uint64_t* d_cnt = (uint64_t*)(d_mu + nd);
  int32_t* d_st = (int32_t*)(d_cnt + CATAPULT_NCOUNTERS);
  uint32_t* d_na = (uint32_t*)(d_st + nd);
  uint32_t* d_nr = d_na + nd;
  const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
  const size_t cb = CATAPULT_NCOUNTERS * sizeof(uint64_t);
  cudaError_t e = cudaMemcpyAsync(d_x, h_x, 4 * nd * sizeof(double), H2D, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_t, h_t, nd * sizeof(double), H2D, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_dt, h_dt, nd * sizeof(double), H2D, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_mu, h_mu, nd * sizeof(double), H2D, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_st, h_status, nd * sizeof(int32_t), H2D, s);
  if (e == cudaSuccess) e = h_nacc ? cudaMemcpyAsync(d_na, h_nacc, nd * sizeof(uint32_t), H2D, s)
                                   : cudaMemsetAsync(d_na, 0, nd * sizeof(uint32_t), s);
  if (e == cudaSuccess) e = h_nrej ? cudaMemcpyAsync(d_nr, h_nrej, nd * sizeof(uint32_t), H2D, s)
                                   : cudaMemsetAsync(d_nr, 0, nd * sizeof(uint32_t), s);
  if (e == cudaSuccess) e = h_counters ? cudaMemcpyAsync(d_cnt, h_counters, cb, H2D, s) : cudaMemsetAsync(d_cnt, 0, cb, s);
  if (e == cudaSuccess) {
    st = catapult_trace_continue(f, p, n, d_x, d_t, d_dt, d_mu, d_st, d_na, d_nr, d_cnt, s);
    if (st == CATAPULT_OK) {
      e = cudaMemcpyAsync(h_x, d_x, 4 * nd * sizeof(double), D2H, s);
      if (e == cudaSuccess) e = cudaMemcpyAsync(h_t, d_t, nd * sizeof(double), D2H, s);
      if (e == cudaSuccess) e = cudaMemcpyAsync(h_dt, d_dt, nd * sizeof(double), D2H, s);
      if (e == cudaSuccess) e = cudaMemcpyAsync(h_mu, d_mu, nd * sizeof(double), D2H, s);
      if (e == cudaSuccess) e = cudaMemcpyAsync(h_status, d_st, nd * sizeof(int32_t), D2H, s);
      if (e == cudaSuccess && h_nacc) e = cudaMemcpyAsync(h_nacc, d_na, nd * sizeof(uint32_t), D2H, s);
      if (e == cudaSuccess && h_nrej) e = cudaMemcpyAsync(h_nrej, d_nr, nd * sizeof(uint32_t), D2H, s);
      if (e == cudaSuccess && h_counters) e = cudaMemcpyAsync(h_counters, d_cnt, cb, D2H, s);
    }
  }
  cudaError_t e2 = cudaStreamSynchronize(s);
  if (st != CATAPULT_OK) return st;
  if (e != cudaSuccess) return cuda_fail(e, "catapult_trace_continue_host copies");
  if (e2 != cudaSuccess) return cuda_fail(e2, "catapult_trace_continue_host");
  return CATAPULT_OK;
}

catapult_status catapult_step_once(const catapult_field* f, const catapult_trace_params* p, int64_t n,
                                   const double* d_x, const double* d_t, const double* d_h, double* d_xnew,
                                   double* d_errratio, double* d_k, void* stream) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (n > 0 && (!d_x || !d_t || !d_h || !d_xnew || !d_errratio || !d_k))
    return fail(CATAPULT_EINVAL, "all array arguments of catapult_step_once are required");
  TraceConst tc;
  int model = 0;
  catapult_status st = make_trace_const(f, p, &tc, &model);
  if (st != CATAPULT_OK) return st;
  st = use_field_on(f, (cudaStream_t)stream);
  if (st != CATAPULT_OK) return st;
  if (n == 0) return CATAPULT_OK;
  TraceArgs a{};
  a.n = n;
  a.x_in = d_x;
  a.x_out = d_xnew;
  a.t_io = const_cast<double*>(d_t);  // read only in this mode
  a.script_h = d_h;
  a.script_r = d_errratio;
  a.kall = d_k;
  cudaStream_t s = (cudaStream_t)stream;
  unsigned long long* queue = nullptr;
  CATAPULT_CUDA_TRY(cudaMallocAsync((void**)&queue, TRACE_SCRATCH_BYTES, s));
  cudaError_t e = cudaMemsetAsync(queue, 0, TRACE_SCRATCH_BYTES, s);
  if (e != cudaSuccess) {
    cudaFreeAsync(queue, s);
    return cuda_fail(e, "cudaMemsetAsync(queue)");
  }
  a.queue = queue;
  st = launch_trace(tc, a, model, 2, s);
  cudaFreeAsync(queue, s);
  return st;
}

catapult_status catapult_estimate(int32_t g_kind, int64_t n, const int32_t* d_status, const double* d_tstop,
                                  const double* d_g_user, double* d_out, double* h_out, void* stream) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (g_kind < 0 || g_kind > 2) return fail(CATAPULT_EINVAL, "g_kind must be 0, 1 or 2");
  if (!d_out) return fail(CATAPULT_EINVAL, "d_out is NULL");
  if (n > 0 && ((g_kind == 0 && !d_status) || (g_kind == 1 && !d_tstop) || (g_kind == 2 && !d_g_user)))
    return fail(CATAPULT_EINVAL, "the array selected by g_kind is NULL");
  catapult_status st = launch_estimate(g_kind, n, d_status, d_tstop, d_g_user, d_out, (cudaStream_t)stream);
  if (st != CATAPULT_OK) return st;
  if (h_out) {
    CATAPULT_CUDA_TRY(cudaMemcpyAsync(h_out, d_out, 4 * sizeof(double), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CATAPULT_CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
  }
  return CATAPULT_OK;
}

catapult_status catapult_measure_lost_energy(const catapult_field* f, const catapult_trace_params* p, int64_t n,
                                             const double* d_xf, const double* d_mu, const int32_t* d_status,
                                             double* d_g, void* stream) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (n > 0 && (!d_xf || !d_mu || !d_status || !d_g)) return fail(CATAPULT_EINVAL, "d_xf, d_mu, d_status and d_g are required");
  TraceConst tc;
  int model = 0;
  catapult_status st = make_trace_const(f, p, &tc, &model);  // validates field and parameters; v_total^2
  if (st != CATAPULT_OK) return st;
  st = use_field_on(f, (cudaStream_t)stream);
  if (st != CATAPULT_OK) return st;
  return launch_lost_energy(f->fc, 2.0 / tc.vtot2, n, d_xf, d_mu, d_status, d_g, (cudaStream_t)stream);
}

catapult_status catapult_exit_histogram(const catapult_field* f, int64_t n, const double* d_xf, const int32_t* d_status,
                                        int32_t nbins0, int32_t nbins1, uint64_t* d_hist, void* stream) {
  if (!f) return fail(CATAPULT_EINVAL, "field is NULL");
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (nbins0 < 1 || nbins1 < 1 || (int64_t)nbins0 * nbins1 > (int64_t)1 << 24)
    return fail(CATAPULT_EINVAL, "nbins0, nbins1 must be >= 1 with at most 2^24 bins in all");
  if (!d_hist || (n > 0 && (!d_xf || !d_status))) return fail(CATAPULT_EINVAL, "d_xf, d_status and d_hist are required");
  catapult_status st = use_device_of(f);  // geometry only: the tables are not read
  if (st != CATAPULT_OK) return st;
  return launch_exit_histogram(f->fc, n, d_xf, d_status, nbins0, nbins1, reinterpret_cast<unsigned long long*>(d_hist),
                               (cudaStream_t)stream);
}

// The estimate without any allocation (include/catapult.h): same validation as catapult_estimate, the size limit and
// the static scratch array are estimate.cu's.
catapult_status catapult_estimate_static(int32_t g_kind, int64_t n, const int32_t* d_status, const double* d_tstop,
                                         const double* d_g_user, double* d_out, void* stream) {
  if (n < 0) return fail(CATAPULT_EINVAL, "n < 0");
  if (g_kind < 0 || g_kind > 2) return fail(CATAPULT_EINVAL, "g_kind must be 0, 1 or 2");
  if (!d_out) return fail(CATAPULT_EINVAL, "d_out is NULL");
  if (n > 0 && ((g_kind == 0 && !d_status) || (g_kind == 1 && !d_tstop) || (g_kind == 2 && !d_g_user)))
    return fail(CATAPULT_EINVAL, "the array selected by g_kind is NULL");
  return launch_estimate_static(g_kind, n, d_status, d_tstop, d_g_user, d_out, (cudaStream_t)stream);
}

catapult_status catapult_trace_launch_shape(const catapult_field* f, const catapult_trace_params* p, int32_t* blocks,
                                            int32_t* threads) {
  if (!blocks || !threads) return fail(CATAPULT_EINVAL, "blocks/threads is NULL");
  TraceConst tc;
  int model = 0;
  catapult_status st = make_trace_const(f, p, &tc, &model);
  if (st != CATAPULT_OK) return st;
  int b = 0, t = 0;
  st = trace_launch_shape(model, f->fc.m == 1 && f->fc.coord == CATAPULT_COORD_BOOZER, (int64_t)1 << 40, &b, &t);
  *blocks = b;
  *threads = t;
  return st;
}

}  // extern "C"
