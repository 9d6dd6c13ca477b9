// Pipeline-stage enumeration over contiguous chain segments ("consecutive layers form a
// pipeline stage", PAPER.md:323-338 1F1B, Table 3 "Opt. Stages"; R27).
//
// A stage is a contiguous segment [a, b) of the chain on its own sub-mesh; the tables handed in are those of the chain
// on that sub-mesh.  The first layer of a segment has no producer inside the stage, so only its node cost and penalty
// count:   f_a[j] = node[a][j] + PEN [mask[a][j] == 0],  f_l[j] = min_i f_{l-1}[i] + T[l][i][j],  C(a, b) = min_j f_{b-1}[j].
//
// segment_optima_kernel: ALL L (L + 1) / 2 segment optima in one pass over the tables.  For a fixed layer l every start
// a < l needs the same tile: F_l[a][.] = F_{l-1}[a][.] (min,+) T[l] is a min-plus product of the (starts x K) state
// matrix with the K x K tile, so a tile is streamed once per block of 16 starts instead of once per start.  One CTA per
// block of 16 consecutive starts; thread (j, g) owns column j of the starts g, g + G, ...; the tile passes through
// shared memory in row blocks; after every layer one warp per start takes min_j and writes C(a, l + 1).
// partition_kernel: DP over the cuts (one CTA, threads over the end position).  segment_strategies_kernel: the optimum
// strategy of each chosen segment with back-pointers (one CTA per stage).
#include "common.cuh"

namespace autoddl {

namespace {

// AB starts per CTA: 16 when there are enough blocks of starts to fill the machine, else 4 (a long single chain: the tiles then
// come from L2 more often, but four times as many SMs share the work and the longest CTA does a quarter of it)
template <int G, int AB>
__global__ void __launch_bounds__(1024) segment_optima_kernel(const int64_t* __restrict__ T, const int64_t* __restrict__ node,
                                                              const uint8_t* __restrict__ mask, int L, int K, int RB,
                                                              int64_t* __restrict__ tri) {
  constexpr int kAB = AB, NA = (AB + G - 1) / G;
  extern __shared__ __align__(16) unsigned char so_smem[];
  int64_t* F = reinterpret_cast<int64_t*>(so_smem);        // [2][kAB][K]
  int64_t* stage = F + 2 * kAB * K;                        // [2][RB][K]: row blocks of the tiles, double buffered (cp.async)
  const int tid = threadIdx.x, nthr = blockDim.x;
  const int j = tid % K, g = tid / K;                      // threads beyond G * K only help with the copies
  const bool worker = g < G;
  const int a0 = blockIdx.x * kAB;
  const int na = L - a0 < kAB ? L - a0 : kAB;              // starts of this block
  for (int x = tid; x < na * (L + 1); x += nthr) tri[(size_t)a0 * (L + 1) + x] = -1;
  // rows r0 .. of tile l -> stage buffer `buf`, asynchronously (8 bytes per request: tiles of an odd K are only 8-byte aligned)
  auto issue = [&](int l, int r0, int buf) {
    const int nr = K - r0 < RB ? K - r0 : RB;
    const int64_t* src = T + (size_t)l * K * K + (size_t)r0 * K;
    int64_t* dst = stage + (size_t)buf * RB * K;
    for (int x = tid; x < nr * K; x += nthr)
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst + x)), "l"(src + x) : "memory");
  };
  int buf = 0;
  if (a0 + 1 < L) issue(a0 + 1, 0, 0);                     // the first tile any start of the block consumes
  asm volatile("cp.async.commit_group;" ::: "memory");
  __syncthreads();
  int cur = 0;
  for (int l = a0; l < L; ++l) {
    int64_t* Fc = F + cur * kAB * K;
    int64_t* Fn = F + (cur ^ 1) * kAB * K;
    int64_t acc[NA];
#pragma unroll
    for (int t = 0; t < NA; ++t) acc[t] = INT64_MAX;
    const int nact = l - a0 < na ? l - a0 : na;            // starts a < l of this block: they consume tile l
    if (nact > 0) {
      for (int r0 = 0; r0 < K; r0 += RB) {
        const int nr = K - r0 < RB ? K - r0 : RB;
        // the next row block (of this tile, or the first of the next tile) travels while this one is consumed
        if (r0 + RB < K) issue(l, r0 + RB, buf ^ 1);
        else if (l + 1 < L) issue(l + 1, 0, buf ^ 1);
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncthreads();
        const int64_t* stg = stage + (size_t)buf * RB * K;
        if (worker) {
          for (int r = 0; r < nr; ++r) {
            const int64_t tv = stg[r * K + j];
#pragma unroll
            for (int t = 0; t < NA; ++t) {
              const int ai = g + G * t;
              if (ai < nact) {
                const int64_t v = Fc[ai * K + r0 + r] + tv;
                if (v < acc[t]) acc[t] = v;
              }
            }
          }
        }
        __syncthreads();                                   // the buffer is free for the copy issued in the next round
        buf ^= 1;
      }
    }
    if (worker) {
#pragma unroll
      for (int t = 0; t < NA; ++t) {
        const int ai = g + G * t;
        if (ai < nact) Fn[ai * K + j] = acc[t];
      }
    }
    if (l - a0 < na && tid < K)                            // the segment that starts at l: node cost + penalty only
      Fn[(l - a0) * K + tid] = node[(size_t)l * K + tid] + (mask[(size_t)l * K + tid] ? 0 : AUTODDL_PEN);
    __syncthreads();
    cur ^= 1;
    // C(a, l + 1) = min_j F[a][j] for every start a <= l of the block: one warp per start
    const int nrec = l - a0 + 1 < na ? l - a0 + 1 : na;
    for (int ai = tid >> 5; ai < nrec; ai += nthr >> 5) {
      int64_t m = INT64_MAX;
      for (int c = tid & 31; c < K; c += 32) {
        const int64_t v = Fn[ai * K + c];
        if (v < m) m = v;
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        const int64_t o = __shfl_xor_sync(0xffffffffu, m, off);
        if (o < m) m = o;
      }
      if ((tid & 31) == 0) tri[(size_t)(a0 + ai) * (L + 1) + l + 1] = m;
    }
    // (the next layer writes the other buffer and its first barrier orders these reads before any overwrite of Fn)
  }
}

__global__ void stage_transfer_kernel(const autoddl_layer* __restrict__ layers, int L, int64_t q, int64_t m, int64_t alpha,
                                      int64_t beta, int64_t* __restrict__ xfer) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= L) return;
  if (b == 0) { xfer[0] = 0; return; }
  const int64_t bytes = layers[b].in_rows * layers[b].in_cols * (int64_t)layers[b].act_bytes;
  xfer[b] = 2 * m * (alpha + (bytes + q - 1) / q * beta);
}

// g_1[b] = c(0, b); g_k[b] = min_a comb(g_{k-1}[a], c(a, b)), smallest a on ties; back-track from g_stages[L]
__global__ void __launch_bounds__(1024) partition_kernel(const int64_t* __restrict__ tri, const int64_t* __restrict__ xfer, int L,
                                                         int stages, int objective, int64_t* __restrict__ gbuf,
                                                         int32_t* __restrict__ argbuf, int64_t* __restrict__ value,
                                                         int32_t* __restrict__ cuts) {
  const int W = L + 1;
  auto c = [&](int a, int b) { return tri[(size_t)a * W + b] + xfer[a] + (b < L ? xfer[b] : 0); };
  for (int x = threadIdx.x; x < (stages + 1) * W; x += blockDim.x) { gbuf[x] = INT64_MAX; argbuf[x] = -1; }
  __syncthreads();
  for (int b = 1 + threadIdx.x; b <= L; b += blockDim.x) { gbuf[W + b] = c(0, b); argbuf[W + b] = 0; }
  __syncthreads();
  for (int k = 2; k <= stages; ++k) {
    for (int b = k + threadIdx.x; b <= L; b += blockDim.x) {
      int64_t best = INT64_MAX;
      int arg = -1;
      for (int a = k - 1; a < b; ++a) {
        const int64_t prev = gbuf[(size_t)(k - 1) * W + a];
        if (prev == INT64_MAX) continue;
        const int64_t cs = c(a, b);
        const int64_t v = objective == 0 ? prev + cs : (prev > cs ? prev : cs);
        if (v < best) { best = v; arg = a; }
      }
      gbuf[(size_t)k * W + b] = best;
      argbuf[(size_t)k * W + b] = arg;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    *value = gbuf[(size_t)stages * W + L];
    cuts[stages] = L;
    for (int k = stages; k >= 1; --k) cuts[k - 1] = argbuf[(size_t)k * W + cuts[k]];
  }
}

// one CTA per stage: chain DP of the segment [cuts[k], cuts[k + 1]) with byte back-pointers in the workspace; thread
// (j, part) scans every fourth row i of column j (increasing i, strict '<': its smallest i), the parts merge by shuffles
__global__ void __launch_bounds__(1024) segment_strategies_kernel(const int64_t* __restrict__ T, const int64_t* __restrict__ node,
                                                                  const uint8_t* __restrict__ mask, int L, int K,
                                                                  const int32_t* __restrict__ cuts, uint8_t* __restrict__ bp,
                                                                  int64_t* __restrict__ seg_cost, int32_t* __restrict__ strategy) {
  constexpr int PARTS = 4;
  __shared__ int64_t f[2][256];
  const int k = blockIdx.x, tid = threadIdx.x, j = tid / PARTS, part = tid % PARTS;
  const int a = cuts[k], b = cuts[k + 1];
  if (a < 0 || b > L || a >= b) return;
  int cur = 0;
  if (tid < K) f[0][tid] = node[(size_t)a * K + tid] + (mask[(size_t)a * K + tid] ? 0 : AUTODDL_PEN);
  __syncthreads();
  for (int l = a + 1; l < b; ++l) {
    const int64_t* col = T + (size_t)l * K * K + (j < K ? j : 0);
    int64_t best = INT64_MAX;
    int ar = 1 << 30;
    if (j < K)
      for (int i = part; i < K; i += PARTS) {
        const int64_t v = f[cur][i] + __ldg(col + (size_t)i * K);
        if (v < best) { best = v; ar = i; }
      }
#pragma unroll
    for (int off = 1; off < PARTS; off <<= 1) {            // (every lane of the warp takes part)
      const int64_t ov = __shfl_xor_sync(0xffffffffu, best, off);
      const int oa = __shfl_xor_sync(0xffffffffu, ar, off);
      if (ov < best || (ov == best && oa < ar)) { best = ov; ar = oa; }
    }
    if (j < K && part == 0) {
      f[cur ^ 1][j] = best;
      bp[(size_t)l * K + j] = (uint8_t)ar;
    }
    __syncthreads();
    cur ^= 1;
  }
  if (tid == 0) {
    int js = 0;
    for (int c = 1; c < K; ++c)
      if (f[cur][c] < f[cur][js]) js = c;
    seg_cost[k] = f[cur][js];
    strategy[b - 1] = js;
    for (int l = b - 1; l > a; --l) strategy[l - 1] = bp[(size_t)l * K + strategy[l]];
  }
}

}  // namespace

int launch_segment_optima(const int64_t* d_T, const int64_t* d_node, const uint8_t* d_mask, int32_t L, int32_t K,
                          int64_t* d_tri, cudaStream_t st) {
  // large tiles of one long chain: 4 starts per CTA (measured: K = 216, L = 480 29 -> 18 ms; small tiles are better off with 16)
  const int AB = K > 64 && (L + 15) / 16 * 2 < device_sm_count() ? 4 : 16;
  const int G = AB == 16 && K <= 64 ? 16 : 4;              // thread groups over the starts of a block
  int threads = (K * G + 31) / 32 * 32;
  if (threads > 1024) threads = 1024;                      // K = 256, G = 4: exactly 1024
  int RB = (int)((92 * 1024) / ((size_t)K * 8));            // rows per stage buffer (two buffers)
  if (RB > K) RB = K;
  if (RB < 1) RB = 1;
  const size_t smem = ((size_t)2 * AB * K + (size_t)2 * RB * K) * 8;
  const int grid = (L + AB - 1) / AB;
  auto go = [&](auto kern) -> int {
    ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid, threads, smem, st>>>(d_T, d_node, d_mask, L, K, RB, d_tri);
    return AUTODDL_OK;
  };
  int rc;
  if (AB == 4) rc = go(segment_optima_kernel<4, 4>);
  else rc = G == 16 ? go(segment_optima_kernel<16, 16>) : go(segment_optima_kernel<4, 16>);
  if (rc) return rc;
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

int launch_stage_transfer(const autoddl_layer* d_layers, int32_t L, int64_t q, int64_t m, int64_t alpha, int64_t beta,
                          int64_t* d_xfer, cudaStream_t st) {
  stage_transfer_kernel<<<(L + 255) / 256, 256, 0, st>>>(d_layers, L, q, m, alpha, beta, d_xfer);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

size_t partition_workspace_bytes(int32_t L, int32_t stages) { return ((size_t)(stages + 1) * (L + 1) * 12 + 255) / 256 * 256 + 256; }

int launch_partition(const int64_t* d_tri, const int64_t* d_xfer, int32_t L, int32_t stages, int32_t objective, void* d_work,
                     int64_t* d_value, int32_t* d_cuts, cudaStream_t st) {
  int64_t* g = (int64_t*)d_work;
  int32_t* arg = (int32_t*)(g + (size_t)(stages + 1) * (L + 1));
  int threads = (L + 32) / 32 * 32;
  if (threads > 1024) threads = 1024;
  partition_kernel<<<1, threads, 0, st>>>(d_tri, d_xfer, L, stages, objective, g, arg, d_value, d_cuts);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

int launch_segment_strategies(const int64_t* d_T, const int64_t* d_node, const uint8_t* d_mask, int32_t L, int32_t K,
                              const int32_t* d_cuts, int32_t stages, uint8_t* d_bp, int64_t* d_seg_cost, int32_t* d_strategy,
                              cudaStream_t st) {
  segment_strategies_kernel<<<stages, (K * 4 + 31) / 32 * 32, 0, st>>>(d_T, d_node, d_mask, L, K, d_cuts, d_bp, d_seg_cost, d_strategy);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
