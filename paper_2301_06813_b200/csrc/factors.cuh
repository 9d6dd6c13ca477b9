// Shared by the kernels that work on the FACTORS of the cost tables (factors.cu: best-response Coordinate Descent;
// chain_dp_scan.cu: chain DP in class space): the layout of a tile's factor block and the class tables.
// Everything has internal linkage (anonymous namespace): each translation unit gets its own copy.
#pragma once

#include "sbp_builder.cuh"

namespace autoddl {

namespace {

template <int D> struct Fac {
  static constexpr int K = Pow<D>::K, NS = Pow<D>::NS, NC = Pow<D>::NC, ES = NS + 1, STRIDE = NC + 1;
  static constexpr int HDR = 8;                            // header words: kind, kind of the previous layer, ...
  static constexpr int FB = (HDR + K + ES * ES + 1) / 2 * 2;   // int64 words per tile (16-byte multiple)
  static constexpr int CS = (2 * ES + 15) / 16 * 16;       // bytes per best-response column of ES 16-bit entries (16-byte multiple)
  static constexpr int N2P = (ES * ES + 1) / 2 * 2;        // words between two ES x ES class matrices (16-byte multiple)
  static constexpr int SQ = (ES + 7) / 16 * 16 + 8;        // row stride of a chunk product Q: = 8 mod 16, see chunk_prefix_kernel
};

// state-vector classes of the signatures per layer kind: A(i) = a_idx (NS if invalid), B(j) = b_idx (NS if invalid)
template <int D>
__device__ __forceinline__ void fill_classes(uint8_t (*acls)[Pow<D>::K], uint8_t (*bcls)[Pow<D>::K], const SigInfo (*sig)[Pow<D>::K],
                                             int tid, int nthr) {
  constexpr int K = Pow<D>::K, NS = Pow<D>::NS;
  for (int x = tid; x < 2 * K; x += nthr) {
    const SigInfo& si = sig[x / K][x % K];
    acls[x / K][x % K] = (uint8_t)si.a_idx;
    bcls[x / K][x % K] = (uint8_t)(si.b_idx >= 0 ? si.b_idx : NS);
  }
}

// per kind: the signatures of every producer class, ascending -- a warp per (kind, class), 32 signatures per ballot
template <int D>
__device__ __forceinline__ void fill_members(uint8_t (*mstart)[Fac<D>::ES + 1], uint8_t (*mlist)[Fac<D>::K],
                                             const uint8_t (*acls)[Fac<D>::K], int tid, int nthr) {
  constexpr int K = Fac<D>::K, ES = Fac<D>::ES;
  const int lane = tid & 31, warp = tid >> 5, nw = nthr >> 5;
  for (int pr = warp; pr < 2 * ES; pr += nw) {
    const int kind = pr / ES, al = pr % ES;
    int n = 0;
    for (int c0 = 0; c0 < K; c0 += 32) n += __popc(__ballot_sync(0xffffffffu, c0 + lane < K && acls[kind][c0 + lane] == al));
    if (lane == 0) mstart[kind][al + 1] = (uint8_t)n;      // (counts for now)
  }
  __syncthreads();
  if (tid < 2) {
    int n = 0;
    mstart[tid][0] = 0;
    for (int al = 0; al < ES; ++al) { n += mstart[tid][al + 1]; mstart[tid][al + 1] = (uint8_t)n; }
  }
  __syncthreads();
  for (int pr = warp; pr < 2 * ES; pr += nw) {
    const int kind = pr / ES, al = pr % ES;
    int n = mstart[kind][al];
    for (int c0 = 0; c0 < K; c0 += 32) {
      const bool mine = c0 + lane < K && acls[kind][c0 + lane] == al;
      const uint32_t m = __ballot_sync(0xffffffffu, mine);
      if (mine) mlist[kind][n + __popc(m & ((1u << lane) - 1))] = (uint8_t)(c0 + lane);
      n += __popc(m);
    }
  }
  __syncthreads();
}

}  // namespace

}  // namespace autoddl
