// Field-table kernels: unique nodes -> per-cell 64-coefficient tables, the
// tricubic test hook and the export in the paper's own row layout.
#include "gc_device.cuh"

namespace catapult {

// One thread per table element.  out[(cell*m + q)*64 + node], node = (a*4+b)*4+c,
// value = nodes[q][3*i0+a][3*i1+b][3*i2+c].  Writes are fully coalesced; the reads of a cell's
// 4-node runs come from L2 (the unique-node array is 64/27 times smaller than the table).
__global__ void __launch_bounds__(256)
field_build_kernel(const double* __restrict__ nodes, double* __restrict__ table, int m, int k0, int k1, int k2) {
  const long long total = (long long)k0 * k1 * k2 * m * 64;
  const long long n1 = 3LL * k1 + 1, n2 = 3LL * k2 + 1, n0 = 3LL * k0 + 1;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total;
       o += (long long)gridDim.x * blockDim.x) {
    const int node = (int)(o & 63);
    const long long cq = o >> 6;
    const int q = (int)(cq % m);
    const long long cell = cq / m;
    const int i2 = (int)(cell % k2);
    const long long r = cell / k2;
    const int i1 = (int)(r % k1);
    const int i0 = (int)(r / k1);
    const int a = node >> 4, b = (node >> 2) & 3, c = node & 3;
    const long long j0 = 3LL * i0 + a, j1 = 3LL * i1 + b, j2 = 3LL * i2 + c;
    table[o] = nodes[(long long)q * n0 * n1 * n2 + (j0 * n1 + j1) * n2 + j2];
  }
}

// test hook: the production evaluation path (group of NL lanes per point, coefficients staged through
// the on-chip cell cache) at arbitrary points
template <int MODEL>
__global__ void __launch_bounds__(ModelTraits<MODEL>::NT, ModelTraits<MODEL>::MINB)
field_eval_kernel(const __grid_constant__ FieldConst f, long long npts, const double* __restrict__ pts,
                  double* __restrict__ out) {
  using MT = ModelTraits<MODEL>;
  extern __shared__ double2 smem[];
  const Group<MT::NL> g;
  CellCache<MODEL> cc;
  cc.init(smem);
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / MT::NL;
  if (i >= npts) return;  // group-uniform
  double u[3], fv[MT::NQ];
  const long long cell = locate<!MT::CART>(f, pts[i], pts[npts + i], pts[2 * npts + i], u);
  tricubic_group<MODEL>(f, g, cc, cell, u, fv);
  if (g.j == 0) {
#pragma unroll
    for (int q = 0; q < MT::NQ; ++q) out[(long long)q * npts + i] = fv[q];
  }
}

// table [cell][q][64] -> rows [(cell*64+node)][q]  (row = node, column = quantity)
__global__ void field_export_rows_kernel(const double* __restrict__ table, double* __restrict__ out, int m,
                                         long long ncells) {
  const long long total = ncells * m * 64;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total;
       o += (long long)gridDim.x * blockDim.x) {
    const int q = (int)(o % m);
    const long long row = o / m;
    const int node = (int)(row & 63);
    const long long cell = row >> 6;
    out[o] = table[(cell * m + q) * 64 + node];
  }
}

static int grid_for(long long total, int threads) {
  long long b = (total + threads - 1) / threads;
  const long long cap = 148LL * 16;
  return (int)(b < 1 ? 1 : (b > cap ? cap : b));
}

catapult_status launch_field_build(const catapult_field_desc& d, const double* d_nodes, double* d_table,
                                   cudaStream_t s) {
  const long long total = (long long)d.ncell[0] * d.ncell[1] * d.ncell[2] * d.nquant * 64;
  field_build_kernel<<<grid_for(total, 256), 256, 0, s>>>(d_nodes, d_table, d.nquant, d.ncell[0], d.ncell[1],
                                                          d.ncell[2]);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

template <int MODEL>
static catapult_status field_eval_one(const FieldConst& fc, int64_t npts, const double* d_pts, double* d_out,
                                      cudaStream_t s) {
  using MT = ModelTraits<MODEL>;
  CATAPULT_CUDA_TRY(cudaFuncSetAttribute(field_eval_kernel<MODEL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)MT::SMEM_BYTES));
  const long long per_block = MT::NT / MT::NL;
  const int blocks = (int)((npts + per_block - 1) / per_block);
  field_eval_kernel<MODEL><<<blocks, MT::NT, MT::SMEM_BYTES, s>>>(fc, npts, d_pts, d_out);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

catapult_status launch_field_eval(const FieldConst& fc, int64_t npts, const double* d_pts, double* d_out,
                                  cudaStream_t s) {
  if (npts == 0) return CATAPULT_OK;
  if (fc.coord == CATAPULT_COORD_BOOZER) return field_eval_one<MODEL_BOOZER_VAC>(fc, npts, d_pts, d_out, s);
  return field_eval_one<MODEL_CART>(fc, npts, d_pts, d_out, s);
}

catapult_status launch_field_export_rows(const FieldConst& fc, int64_t ncells, double* d_out, cudaStream_t s) {
  const long long total = ncells * fc.m * 64;
  field_export_rows_kernel<<<grid_for(total, 256), 256, 0, s>>>(fc.table, d_out, fc.m, ncells);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

}  // namespace catapult
