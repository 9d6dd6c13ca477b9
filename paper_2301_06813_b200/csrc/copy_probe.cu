// Device-to-device copy used by bench.py to measure the HBM copy bandwidth in the same run.
// One block per contiguous 8 KB chunk (non-persistent: neighbouring blocks stream neighbouring DRAM pages), two
// 16-byte loads in flight per thread.  Measured on B200: 6.8 TB/s read + write (a persistent grid-stride loop over the
// same data reaches 5.8 TB/s, cudaMemcpyAsync 6.5 TB/s).
#include "common.cuh"

namespace autoddl {

namespace {

constexpr int kU = 2;

__global__ void __launch_bounds__(256) copy_probe_kernel(const int4* __restrict__ src, int4* __restrict__ dst, size_t n) {
  const size_t base = (size_t)blockIdx.x * (256 * kU) + threadIdx.x;
  int4 v[kU];
#pragma unroll
  for (int u = 0; u < kU; ++u)
    if (base + u * 256 < n) v[u] = src[base + u * 256];
#pragma unroll
  for (int u = 0; u < kU; ++u)
    if (base + u * 256 < n) dst[base + u * 256] = v[u];
}

}  // namespace

int launch_copy_probe(const void* src, void* dst, size_t bytes, cudaStream_t st) {
  const size_t n = bytes / 16;
  const size_t blocks = (n + 256 * kU - 1) / (256 * kU);
  if (blocks > 0x7fffffffull) { set_error("copy_probe: too many bytes"); return AUTODDL_EINVAL; }
  copy_probe_kernel<<<(unsigned)blocks, 256, 0, st>>>((const int4*)src, (int4*)dst, n);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
