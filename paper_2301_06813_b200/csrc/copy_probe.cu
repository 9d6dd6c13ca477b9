// Device-to-device copy used by bench.py to measure the HBM copy bandwidth in the same run.
#include "common.cuh"

namespace autoddl {

namespace {

__global__ void __launch_bounds__(256) copy_probe_kernel(const int4* __restrict__ src, int4* __restrict__ dst, size_t n) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (; i + 3 * stride < n; i += 4 * stride) {        // four independent 16-byte loads in flight
    const int4 a = __ldcs(src + i), b = __ldcs(src + i + stride), c = __ldcs(src + i + 2 * stride),
               d = __ldcs(src + i + 3 * stride);
    __stcs(dst + i, a);
    __stcs(dst + i + stride, b);
    __stcs(dst + i + 2 * stride, c);
    __stcs(dst + i + 3 * stride, d);
  }
  for (; i < n; i += stride) __stcs(dst + i, __ldcs(src + i));
}

}  // namespace

int launch_copy_probe(const void* src, void* dst, size_t bytes, cudaStream_t st) {
  int dev = 0, sms = 148;
  ADL_CUDA_CHECK(cudaGetDevice(&dev));
  ADL_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const size_t n = bytes / 16;
  size_t want = (n + 255) / 256;
  const int grid = (int)(want < (size_t)sms * 8 ? want : (size_t)sms * 8);
  copy_probe_kernel<<<grid, 256, 0, st>>>((const int4*)src, (int4*)dst, n);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
