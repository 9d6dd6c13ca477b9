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

// Store-only probe with the ADDRESS PATTERN of the fused table writer (fused_chain.cu): one warp per chain walks the chain's
// tiles in order and writes each tile (cells int64, a multiple of 2) with 16-byte streaming stores, 512 contiguous bytes per
// warp instruction; one CTA of 28 warps per SM.  No arithmetic: what it reaches is the ceiling of that write pattern.
__global__ void __launch_bounds__(896, 1) store_probe_kernel(int64_t* __restrict__ T, int Bp, int L, int cells) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
  for (int p = warp * gridDim.x + blockIdx.x; p < Bp; p += gridDim.x * W)
    for (int l = 0; l < L; ++l) {
      longlong2* o = reinterpret_cast<longlong2*>(T + ((size_t)p * L + l) * cells);
      const longlong2 v = make_longlong2(p, l);
      for (int x = lane; x < cells / 2; x += 32) __stcs(o + x, v);
    }
}

}  // namespace

int launch_store_probe(int64_t* d_T, int32_t Bp, int32_t L, int32_t cells, cudaStream_t st) {
  const int sms = device_sm_count();
  store_probe_kernel<<<Bp < sms ? Bp : sms, 896, 0, st>>>(d_T, Bp, L, cells);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

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
