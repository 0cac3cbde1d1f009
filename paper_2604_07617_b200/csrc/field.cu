// Field-table kernels: unique nodes -> per-cell 64-coefficient tables, the
// tricubic test hook and the export of nodal rows in the paper's own layout.
#include "gc_device.cuh"

namespace catapult {

// ---- double-double helpers (the basis change is done in ~106-bit arithmetic) ---------------------------
struct dd {
  double hi, lo;
};
__device__ __forceinline__ dd dd_norm(double s, double e) {  // |e| <= |s|
  const double h = s + e;
  return dd{h, e - (h - s)};
}
__device__ __forceinline__ dd dd_add(dd x, dd y) {
  const double s = x.hi + y.hi;
  const double bb = s - x.hi;
  const double e = ((x.hi - (s - bb)) + (y.hi - bb)) + (x.lo + y.lo);
  return dd_norm(s, e);
}
__device__ __forceinline__ dd dd_neg(dd x) { return dd{-x.hi, -x.lo}; }
__device__ __forceinline__ dd dd_mul(dd x, double m) {  // m a small integer or a power of two
  const double p = x.hi * m;
  const double e = fma(x.hi, m, -p) + x.lo * m;
  return dd_norm(p, e);
}

// Nodal values f0..f3 at u = 0, 1/3, 2/3, 1 -> coefficients of 1, w, w^2, w^3 with w = 2u - 1.
// The matrix is [-1 9 9 -1; 1 -27 27 -1; 9 -9 -9 9; -9 27 -27 9] / 16 (exact small integers).
__device__ __forceinline__ void nodal_to_monomial(dd& f0, dd& f1, dd& f2, dd& f3) {
  const dd A = dd_add(f1, f2), S = dd_add(f0, f3);
  const dd D = dd_add(f2, dd_neg(f1)), E = dd_add(f3, dd_neg(f0));
  const dd c0 = dd_mul(dd_add(dd_mul(A, 9.0), dd_neg(S)), 0.0625);
  const dd c1 = dd_mul(dd_add(dd_mul(D, 27.0), dd_neg(E)), 0.0625);
  const dd c2 = dd_mul(dd_add(S, dd_neg(A)), 0.5625);
  const dd c3 = dd_mul(dd_add(dd_mul(E, 9.0), dd_neg(dd_mul(D, 27.0))), 0.0625);
  f0 = c0;
  f1 = c1;
  f2 = c2;
  f3 = c3;
}

// One thread per (cell, quantity): gathers the 4x4x4 nodal block nodes[q][3*i0+a][3*i1+b][3*i2+c] (shared faces
// are read by both neighbours), changes basis along the three axes, writes 512 contiguous bytes
// table[(cell*m + q)*64 + coef_pos(boozer, p0, p1, p2)] (gc_device.cuh: coefficient of w0^p0 w1^p1 w2^p2; register
// half first, shared half second).  The thread of (cell 0, quantity 0) also copies the first node of column 0
// (|B| on the axis for a Boozer grid) to *node0: DESIGN.md S3's default step length needs it.
__global__ void __launch_bounds__(128)
field_build_kernel(const double* __restrict__ nodes, double* __restrict__ table, double* __restrict__ node0, int m,
                   int k0, int k1, int k2, int boozer) {
  const long long total = (long long)k0 * k1 * k2 * m;
  const long long n1 = 3LL * k1 + 1, n2 = 3LL * k2 + 1, n0 = 3LL * k0 + 1;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total;
       o += (long long)gridDim.x * blockDim.x) {
    const int q = (int)(o % m);
    const long long cell = o / m;
    const int i2 = (int)(cell % k2);
    const long long r = cell / k2;
    const int i1 = (int)(r % k1);
    const int i0 = (int)(r / k1);
    dd v[64];
    const double* base = nodes + (long long)q * n0 * n1 * n2;
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = 0; b < 4; ++b)
#pragma unroll
        for (int c = 0; c < 4; ++c)
          v[(a * 4 + b) * 4 + c] = dd{base[((3LL * i0 + a) * n1 + (3LL * i1 + b)) * n2 + (3LL * i2 + c)], 0.0};
#pragma unroll
    for (int stride = 1; stride <= 16; stride *= 4) {
#pragma unroll
      for (int g = 0; g < 16; ++g) {
        // the 16 lines along this axis: index = lo + hi*4*stride, lo in [0,stride), hi in [0,16/stride)
        const int e0 = (g % stride) + (g / stride) * 4 * stride;
        nodal_to_monomial(v[e0], v[e0 + stride], v[e0 + 2 * stride], v[e0 + 3 * stride]);
      }
    }
    double* dst = table + o * 64;
    if (boozer) {
#pragma unroll
      for (int e = 0; e < 64; ++e) dst[coef_pos(true, e >> 4, (e >> 2) & 3, e & 3)] = v[e].hi;  // hi = fl(hi + lo)
    } else {
#pragma unroll
      for (int e = 0; e < 64; ++e) dst[coef_pos(false, e >> 4, (e >> 2) & 3, e & 3)] = v[e].hi;
    }
    if (o == 0) *node0 = nodes[0];
  }
}

// test hook: tricubic values of all quantities at arbitrary points with the production locate and
// contraction functions, coefficients read straight from the table
template <bool BOOZER>
__global__ void __launch_bounds__(128)
field_eval_kernel(const __grid_constant__ FieldConst f, long long npts, const double* __restrict__ pts,
                  double* __restrict__ out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npts) return;
  using AX = AxisRoles<BOOZER>;
  double w[3];
  const int cell = locate<BOOZER>(f, pts[i], pts[npts + i], pts[2 * npts + i], w);
  for (int q = 0; q < f.m; ++q) {
    const double* src = f.table + ((long long)cell * f.m + q) * 64;
    out[(long long)q * npts + i] = horner64(
        [&](int e, double& f0, double& f1, double& f2, double& f3) { ldg_f64x4(src + e, f0, f1, f2, f3); },
        w[AX::LAST], w[AX::SECOND], w[AX::FIRST]);
  }
}

// test hook: nodal values recovered from the table in the paper's row layout (row = node,
// column = quantity): out[(cell*64+node)*m + q] = polynomial of (cell,q) at the in-cell node (a,b,c),
// w = -1, -1/3, 1/3, 1.  Equal to the input nodes up to the rounding of the stored coefficients.
template <bool BOOZER>
__global__ void field_export_rows_kernel(const double* __restrict__ table, double* __restrict__ out, int m,
                                         long long ncells) {
  using AX = AxisRoles<BOOZER>;
  const long long total = ncells * m * 64;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total;
       o += (long long)gridDim.x * blockDim.x) {
    const int q = (int)(o % m);
    const long long row = o / m;
    const int node = (int)(row & 63);
    const long long cell = row >> 6;
    const double* src = table + (cell * m + q) * 64;
    const double w[3] = {((node >> 4) * 2 - 3) * (1.0 / 3.0), (((node >> 2) & 3) * 2 - 3) * (1.0 / 3.0),
                         ((node & 3) * 2 - 3) * (1.0 / 3.0)};
    out[o] = horner64(
        [&](int e, double& f0, double& f1, double& f2, double& f3) { ldg_f64x4(src + e, f0, f1, f2, f3); },
        w[AX::LAST], w[AX::SECOND], w[AX::FIRST]);
  }
}

static int grid_for(long long total, int threads) {
  long long b = (total + threads - 1) / threads;
  const long long cap = 148LL * 16;
  return (int)(b < 1 ? 1 : (b > cap ? cap : b));
}

catapult_status launch_field_build(const catapult_field_desc& d, const double* d_nodes, double* d_table,
                                   double* d_node0, cudaStream_t s) {
  const long long total = (long long)d.ncell[0] * d.ncell[1] * d.ncell[2] * d.nquant;
  field_build_kernel<<<grid_for(total, 128), 128, 0, s>>>(d_nodes, d_table, d_node0, d.nquant, d.ncell[0], d.ncell[1],
                                                          d.ncell[2], d.coord == CATAPULT_COORD_BOOZER);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

catapult_status launch_field_eval(const FieldConst& fc, int64_t npts, const double* d_pts, double* d_out,
                                  cudaStream_t s) {
  if (npts == 0) return CATAPULT_OK;
  const int blocks = (int)((npts + 127) / 128);
  if (fc.coord == CATAPULT_COORD_BOOZER) field_eval_kernel<true><<<blocks, 128, 0, s>>>(fc, npts, d_pts, d_out);
  else field_eval_kernel<false><<<blocks, 128, 0, s>>>(fc, npts, d_pts, d_out);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

catapult_status launch_field_export_rows(const FieldConst& fc, int64_t ncells, double* d_out, cudaStream_t s) {
  const long long total = ncells * fc.m * 64;
  if (fc.coord == CATAPULT_COORD_BOOZER)
    field_export_rows_kernel<true><<<grid_for(total, 256), 256, 0, s>>>(fc.table, d_out, fc.m, ncells);
  else
    field_export_rows_kernel<false><<<grid_for(total, 256), 256, 0, s>>>(fc.table, d_out, fc.m, ncells);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

}  // namespace catapult
