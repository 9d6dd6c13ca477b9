// Best of the Coordinate Descent starts (at every fixed point "the algorithm records the best strategy
// and begins anew with a different initial guess"; R10): per problem the start with the smallest cost, the
// smallest start index on ties.  One warp per problem, lexicographic (cost, start) minimum with warp shuffles.
#include "common.cuh"

namespace autoddl {

namespace {

__global__ void __launch_bounds__(256) best_of_starts_kernel(const int64_t* __restrict__ cost, int Bp, int S,
                                                              int64_t* __restrict__ best_cost, int32_t* __restrict__ best_start) {
  const int p = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (p >= Bp) return;
  const int64_t* c = cost + (size_t)p * S;
  int64_t bv = INT64_MAX;
  int bi = INT32_MAX;
  for (int s = lane; s < S; s += 32) {                     // ascending s per lane: strict '<' keeps the first
    const int64_t v = c[s];
    if (v < bv || bi == INT32_MAX) { bv = v; bi = s; }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
    if (oi != INT32_MAX && (bi == INT32_MAX || ov < bv || (ov == bv && oi < bi))) { bv = ov; bi = oi; }
  }
  if (lane == 0) {
    best_cost[p] = bv;
    best_start[p] = bi;
  }
}

}  // namespace

int launch_best_of_starts(const int64_t* d_cost, int32_t Bp, int32_t S, int64_t* d_best_cost, int32_t* d_best_start,
                          cudaStream_t st) {
  const int wpb = 8;
  best_of_starts_kernel<<<(Bp + wpb - 1) / wpb, wpb * 32, 0, st>>>(d_cost, Bp, S, d_best_cost, d_best_start);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
