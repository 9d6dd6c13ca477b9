// alpha-beta calibration: least-squares (alpha, beta) from N timed collectives.
//
// Measurement i (kind, p, n bytes, time t) gives one row of the linear system of Table 2
//   t_i = A_i alpha + B_i beta,   AllGather / ReduceScatter: (p-1, (p-1)/p n), AllReduce: (2p-1, 2 (p-1)/p n),
//                                 AlltoAll: (p-1, n).
// The normal equations need five sums (AA, AB, BB, At, Bt).  B is ~1e9 times A, so both columns are scaled to unit
// maximum first (pass 1: max |A|, max |B|); pass 2 accumulates the scaled sums in fp64 with a fixed grid and a
// fixed reduction tree (deterministic), pass 3 solves the 2 x 2 system by Cramer's rule and unscales.
// HBM-bound: 24 bytes read per measurement per pass.
#include "common.cuh"

namespace autoddl {

namespace {

constexpr int FIT_BLOCK = 256, FIT_GRID_MAX = 592;

__device__ __forceinline__ void design_row(int kind, int p, int64_t n, double& A, double& B) {
  const double pd = (double)p, nd = (double)n;
  if (kind == 2) { A = 2.0 * pd - 1.0; B = 2.0 * (pd - 1.0) / pd * nd; }        // AllReduce
  else if (kind == 3) { A = pd - 1.0; B = nd; }                                 // AlltoAll
  else { A = pd - 1.0; B = (pd - 1.0) / pd * nd; }                              // AllGather, ReduceScatter
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, off));
  return v;
}

// pass 1: per-block max |A|, max |B|  ->  part[block][0..1]
__global__ void __launch_bounds__(FIT_BLOCK)
fit_max_kernel(const int32_t* __restrict__ kind, const int32_t* __restrict__ p, const int64_t* __restrict__ nbytes,
               int64_t N, double* __restrict__ part) {
  __shared__ double sh[2][FIT_BLOCK / 32];
  double ma = 0.0, mb = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * FIT_BLOCK + threadIdx.x; i < N; i += (int64_t)gridDim.x * FIT_BLOCK) {
    double A, B;
    design_row(kind[i], p[i], nbytes[i], A, B);
    ma = fmax(ma, fabs(A));
    mb = fmax(mb, fabs(B));
  }
  ma = warp_max(ma);
  mb = warp_max(mb);
  if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = ma; sh[1][threadIdx.x >> 5] = mb; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < FIT_BLOCK / 32; ++w) { ma = fmax(ma, sh[0][w]); mb = fmax(mb, sh[1][w]); }
    part[2 * blockIdx.x] = ma;
    part[2 * blockIdx.x + 1] = mb;
  }
}

// pass 2: scaled sums per block  ->  sums[block][0..4]
__global__ void __launch_bounds__(FIT_BLOCK)
fit_sum_kernel(const int32_t* __restrict__ kind, const int32_t* __restrict__ p, const int64_t* __restrict__ nbytes,
               const double* __restrict__ t, int64_t N, const double* __restrict__ maxpart, int nmax,
               double* __restrict__ sums) {
  __shared__ double sh[5][FIT_BLOCK / 32];
  // the scales: max over the blocks' maxima, found by the whole block (max is exact: any order gives the same value)
  double ma = 0.0, mb = 0.0;
  for (int k = threadIdx.x; k < nmax; k += FIT_BLOCK) { ma = fmax(ma, maxpart[2 * k]); mb = fmax(mb, maxpart[2 * k + 1]); }
  ma = warp_max(ma);
  mb = warp_max(mb);
  if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = ma; sh[1][threadIdx.x >> 5] = mb; }
  __syncthreads();
  ma = mb = 0.0;
  for (int w = 0; w < FIT_BLOCK / 32; ++w) { ma = fmax(ma, sh[0][w]); mb = fmax(mb, sh[1][w]); }
  __syncthreads();                                         // sh is reused for the sums below
  const double ia = ma > 0.0 ? 1.0 / ma : 0.0, ib = mb > 0.0 ? 1.0 / mb : 0.0;
  double s[5] = {0, 0, 0, 0, 0};
  for (int64_t i = (int64_t)blockIdx.x * FIT_BLOCK + threadIdx.x; i < N; i += (int64_t)gridDim.x * FIT_BLOCK) {
    double A, B;
    design_row(kind[i], p[i], nbytes[i], A, B);
    A *= ia;
    B *= ib;
    const double ti = t[i];
    s[0] += A * A; s[1] += A * B; s[2] += B * B; s[3] += A * ti; s[4] += B * ti;
  }
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const double v = warp_sum(s[q]);
    if ((threadIdx.x & 31) == 0) sh[q][threadIdx.x >> 5] = v;
  }
  __syncthreads();
  if (threadIdx.x < 5) {
    double v = 0.0;
    for (int w = 0; w < FIT_BLOCK / 32; ++w) v += sh[threadIdx.x][w];
    sums[5 * blockIdx.x + threadIdx.x] = v;
  }
}

// pass 3: one block adds the block sums in a fixed order (thread k takes blocks k, k + 256, ..; then a fixed tree), solves the
// 2 x 2 normal equations, unscales.  out = {alpha, beta}
__global__ void __launch_bounds__(FIT_BLOCK) fit_solve_kernel(const double* __restrict__ maxpart, const double* __restrict__ sums,
                                                              int nblocks, double* __restrict__ out) {
  __shared__ double sh[7][FIT_BLOCK / 32];
  double v[7] = {0, 0, 0, 0, 0, 0, 0};                     // ma, mb, five sums
  for (int k = threadIdx.x; k < nblocks; k += FIT_BLOCK) {
    v[0] = fmax(v[0], maxpart[2 * k]);
    v[1] = fmax(v[1], maxpart[2 * k + 1]);
    for (int q = 0; q < 5; ++q) v[2 + q] += sums[5 * k + q];
  }
  v[0] = warp_max(v[0]);
  v[1] = warp_max(v[1]);
#pragma unroll
  for (int q = 2; q < 7; ++q) v[q] = warp_sum(v[q]);
  if ((threadIdx.x & 31) == 0)
    for (int q = 0; q < 7; ++q) sh[q][threadIdx.x >> 5] = v[q];
  __syncthreads();
  if (threadIdx.x != 0) return;
  double ma = 0.0, mb = 0.0, s[5] = {0, 0, 0, 0, 0};
  for (int w = 0; w < FIT_BLOCK / 32; ++w) {
    ma = fmax(ma, sh[0][w]);
    mb = fmax(mb, sh[1][w]);
    for (int q = 0; q < 5; ++q) s[q] += sh[2 + q][w];
  }
  const double det = s[0] * s[2] - s[1] * s[1];
  double a = 0.0, b = 0.0;
  if (det != 0.0) {
    a = (s[3] * s[2] - s[1] * s[4]) / det;
    b = (s[0] * s[4] - s[1] * s[3]) / det;
  }
  out[0] = ma > 0.0 ? a / ma : 0.0;
  out[1] = mb > 0.0 ? b / mb : 0.0;
}

}  // namespace

size_t fit_workspace_bytes() { return (size_t)FIT_GRID_MAX * 7 * sizeof(double); }

int launch_fit_alpha_beta(const int32_t* d_kind, const int32_t* d_p, const int64_t* d_bytes, const double* d_time,
                          int64_t N, double* d_out, double* d_work, cudaStream_t st) {
  int64_t nb = (N + FIT_BLOCK - 1) / FIT_BLOCK;
  const int grid = (int)(nb < FIT_GRID_MAX ? nb : FIT_GRID_MAX);
  double* maxpart = d_work;
  double* sums = d_work + 2 * FIT_GRID_MAX;
  fit_max_kernel<<<grid, FIT_BLOCK, 0, st>>>(d_kind, d_p, d_bytes, N, maxpart);
  fit_sum_kernel<<<grid, FIT_BLOCK, 0, st>>>(d_kind, d_p, d_bytes, d_time, N, maxpart, grid, sums);
  fit_solve_kernel<<<1, FIT_BLOCK, 0, st>>>(maxpart, sums, grid, d_out);
  count_launch(3);
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
