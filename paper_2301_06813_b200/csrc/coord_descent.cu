// (a3) Multi-start Coordinate Descent (R10) for sm_100a.
//
// One block (one warp) per (problem, start).  A sweep visits l = 0..L-1 in order; the update of layer l
//   s_l <- smallest-index argmin_c  T[l][s_{l-1}][c] + T[l+1][c][s_{l+1}]
// reads one contiguous row and one strided column of the tables; lanes take candidates c, the minimum
// and its lowest index are found with warp shuffles on the pair (cost, index).
//
// An update whose two neighbours have not changed since the layer was last updated would recompute the
// same argmin (it is a deterministic function of (s_{l-1}, s_{l+1})), so it is skipped: a per-layer
// dirty flag is set whenever a neighbour's signature changes.  The trajectory, the sweep count and the
// result are identical to the plain algorithm; only redundant table reads disappear.
#include "common.cuh"

namespace autoddl {

namespace {

// smallest (value, index) over the warp.  Fast path when every lane holds a value in [0, 2^55) and an index below 256: the
// key value * 256 + index is reduced as two 32-bit halves with redux.sync (the low half only among the lanes that hold the
// smallest high half); otherwise the shuffle butterfly.  Both are exact.
__device__ __forceinline__ void warp_argmin(int64_t& bv, int& bi) {
  if (__all_sync(0xffffffffu, (uint64_t)bv < (1ull << 55) && (unsigned)bi < 256u)) {
    const uint64_t key = ((uint64_t)bv << 8) | (uint32_t)bi;
    const uint32_t hi = (uint32_t)(key >> 32), lo = (uint32_t)key;
    const uint32_t mh = __reduce_min_sync(0xffffffffu, hi);
    const uint32_t ml = __reduce_min_sync(0xffffffffu, hi == mh ? lo : 0xffffffffu);
    const uint64_t m = ((uint64_t)mh << 32) | ml;
    bv = (int64_t)(m >> 8);
    bi = (int)(m & 255);
    return;
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
    if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
  }
}

// 8-byte read-only load that asks L2 to fetch only a 64-byte granule (a column gather touches one element per
// 288-byte row, so anything wider is wasted DRAM traffic)
__device__ __forceinline__ int64_t ldg_narrow(const int64_t* p) {
  int64_t v;
  asm volatile("ld.global.nc.L2::64B.b64 %0, [%1];" : "=l"(v) : "l"(p));
  return v;
}

// RESUME: the first sweep -- or the first two (prev != NULL: the strategies after sweep 1) -- were run elsewhere (the fused
// kernel does them from the tile factors in shared memory) and the result of the last one is in `strategy`.  A layer is
// dirty iff its right neighbour changed in the last sweep done (a layer is touched once per sweep and sees its left
// neighbour's new value); the sweep count starts at 1 or 2; a sweep that changed nothing ends the descent -- so if sweep 1
// changed nothing the answer is its result with a count of 1, whatever was run after it.
// SBPROWS: the tables were built by this library (autoddl_search, or d_T == NULL), so rows of a tile whose producer
// signatures agree up to the per-level classes {0}, {1}, {3}, {2, 4, 5} are identical (signatures 2, 4, 5 all output P,
// or are all invalid for ATTN: DESIGN.md R1): the column gather reads the class representative's row, and candidates
// of one class share one 64-byte granule -- 16 instead of 36 at K = 36.  Values, hence results, are unchanged.
// KT = 0: K is a launch parameter (any K <= 256: the mixed-radix signature spaces of four / five mesh levels, R26)
template <int KT, bool RESUME, bool SBPROWS>
__global__ void __launch_bounds__(32) coord_descent_kernel(const int64_t* __restrict__ T, int Krt, int L, int S,
                                                           const int32_t* __restrict__ init, int max_sweeps,
                                                           int64_t* __restrict__ cost, int32_t* __restrict__ strategy,
                                                           int32_t* __restrict__ sweeps, const int32_t* __restrict__ prev) {
  extern __shared__ __align__(16) unsigned char smem[];
  int32_t* s = reinterpret_cast<int32_t*>(smem);            // [L]
  uint8_t* dirty = reinterpret_cast<uint8_t*>(s + L);        // [L]

  const int lane = threadIdx.x;
  const size_t ps = blockIdx.x;
  const size_t p = ps / S;
  const int K = KT ? KT : Krt;
  const int64_t* Tp = T + p * (size_t)L * K * K;
  constexpr int NCAND = KT ? (KT + 31) / 32 : 8;
  int rep[NCAND];                                          // row that holds candidate c's column value
#pragma unroll
  for (int q = 0; q < NCAND; ++q) {
    const int c = 32 * q + lane;
    int r = 0, pw = 1, x = c;
    if (SBPROWS) {
      for (int d = 0; d < 3 && pw < K; ++d) {              // base-6 digits, least significant first
        const int dig = x % 6;
        x /= 6;
        r += (dig < 4 ? dig : 2) * pw;
        pw *= 6;
      }
    } else {
      r = c;
    }
    rep[q] = r;
  }

  int nsweeps = 0;
  bool resume_done = false;
  if (RESUME) {
    bool any1 = false, any2 = false;                       // sweep 1 / sweep 2 changed something
    for (int l = lane; l < L; l += 32) {
      const int s0 = init[ps * L + l], s1 = prev ? prev[ps * L + l] : strategy[ps * L + l];
      any1 |= s1 != s0;
      if (prev) any2 |= strategy[ps * L + l] != s1;
    }
    any1 = __any_sync(0xffffffffu, any1);
    any2 = __any_sync(0xffffffffu, any2);
    const bool two = prev != nullptr && any1 && max_sweeps > 1;     // sweep 2 counts
    for (int l = lane; l < L; l += 32) {
      const int32_t* last = two || !prev ? strategy : prev;         // the state the descent stands at
      const int32_t* before = two ? prev : init;                    // the state one sweep earlier
      s[l] = last[ps * L + l];
      dirty[l] = (l + 1 < L && last[ps * L + l + 1] != before[ps * L + l + 1]) ? 1 : 0;
    }
    nsweeps = two ? 2 : 1;
    resume_done = !any1 || max_sweeps <= 1 || (two && (!any2 || max_sweeps <= 2));
  } else {
    for (int l = lane; l < L; l += 32) {
      s[l] = init[ps * L + l];
      dirty[l] = 1;
    }
  }
  __syncwarp();

  // The column T[l+1][.][s_{l+1}] of an update is known long before the update runs (s_{l+1} is not touched before
  // layer l+1's own turn), the row T[l][s_{l-1}][.] only when layer l-1 is done.  So the column gather of the NEXT dirty
  // layer is issued before the argmin of the current one and only the contiguous row read stays on the dependent
  // chain.  If the current update changes its layer, layer l+1 becomes dirty and runs next: a prefetch made for a
  // later layer is then dropped.  (Reading the next row speculatively as well was measured and costs more than it
  // saves, on the batched config and with one model and many starts alike: 191 -> 211 us on config 3, 1,328 -> 1,486 us
  // on config 5.)
  auto next_dirty = [&](int from) {                        // 32 flags per step: lane i looks at layer base + i
    for (int base = from & ~31; base < L; base += 32) {
      const int l = base + lane;
      const unsigned m = __ballot_sync(0xffffffffu, l >= from && l < L && dirty[l]);
      if (m) return base + __ffs(m) - 1;
    }
    return L;
  };
  auto load_row = [&](int l, int64_t (&rv)[NCAND]) {
    const int64_t* row = Tp + ((size_t)l * K + (l > 0 ? s[l - 1] : 0)) * K;
#pragma unroll
    for (int q = 0; q < NCAND; ++q) {
      const int c = 32 * q + lane;
      rv[q] = c < K ? __ldg(row + c) : 0;
    }
  };
  auto load_col = [&](int l, int64_t (&cv)[NCAND]) {
    const bool has_right = l < L - 1;
    const int64_t* col = Tp + (size_t)(l + 1) * K * K + (has_right ? s[l + 1] : 0);
#pragma unroll
    for (int q = 0; q < NCAND; ++q) {
      const int c = 32 * q + lane;
      cv[q] = (has_right && c < K) ? ldg_narrow(col + (size_t)rep[q] * K) : 0;
    }
  };
  for (; !resume_done;) {
    bool changed = false;
    int l = next_dirty(0);
    int64_t cvp[NCAND];                                      // prefetched column of layer pf
    int pf = -1;
    if (l < L) { load_col(l, cvp); pf = l; }
    while (l < L) {
      int64_t cv[NCAND], rv[NCAND];
      if (pf == l) {
#pragma unroll
        for (int q = 0; q < NCAND; ++q) cv[q] = cvp[q];
      } else {
        load_col(l, cv);
      }
      load_row(l, rv);
      int l2 = next_dirty(l + 1);
      pf = -1;
      if (l2 < L) { load_col(l2, cvp); pf = l2; }            // in flight during this layer's argmin
      int64_t bv = INT64_MAX;
      int bi = K;
#pragma unroll
      for (int q = 0; q < NCAND; ++q) {
        const int c = 32 * q + lane;
        if (c < K) {
          const int64_t g = rv[q] + cv[q];
          if (g < bv) { bv = g; bi = c; }
        }
      }
      warp_argmin(bv, bi);
      const int old = s[l];
      __syncwarp();
      if (lane == 0) {
        dirty[l] = 0;
        if (bi != old) {
          s[l] = bi;
          if (l > 0) dirty[l - 1] = 1;
          if (l < L - 1) dirty[l + 1] = 1;
        }
      }
      __syncwarp();
      if (bi != old) {
        changed = true;
        if (l + 1 < L) l2 = l + 1;                           // now dirty: it runs next (its column prefetch exists iff pf == l + 1)
      }
      l = l2;
    }
    ++nsweeps;
    if (!changed || nsweeps >= max_sweeps) break;
  }

  // Cost(s) = sum_l T[l][s_{l-1}][s_l]
  int64_t acc = 0;
  for (int l = lane; l < L; l += 32) {
    const int left = l > 0 ? s[l - 1] : 0;
    acc += ldg_narrow(Tp + ((size_t)l * K + left) * K + s[l]);
    strategy[ps * L + l] = s[l];
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
  if (lane == 0) {
    cost[ps] = acc;
    sweeps[ps] = nsweeps;
  }
}

// The SWEEPS of one start run side by side (chains of at least 8 layers).  Update (k, l) -- sweep k, layer l --
// reads s_{l-1} as sweep k left it and s_{l+1} as sweep k-1 left it, so sweep k may follow sweep k-1 two layers behind: warp w
// of the block runs sweeps w+1, w+1+W, ... on the one state array in shared memory.  That is the plain loop nest in another
// order: every update sees the operands it sees there, so trajectory, result and sweep count are the sequential algorithm's.
// The state of a layer is ONE word -- the sweep that visited it last << 16 | whether that visit changed it << 15 | s_l --
// so the word a follower waits for (layer l+1 tagged k-1) carries the operand itself and the leading sweep never fences.
// A layer is re-evaluated in sweep k only if s_{l-1} changed in sweep k or s_{l+1} in sweep k-1: the dirty rule above.  The
// first sweep that changes nothing ends the descent (stop); sweeps already under way behind it are no-ops by then.
constexpr int kWaveWarps = 8;
constexpr int kWaveWideBlocks = 296;                       // up to two starts per SM: eight sweeps of a start in flight, else four
constexpr int kWaveMaxBlocks = 2048;                       // RESUME beyond that: one warp per start (the few updates left gain nothing)
// RESUME: as in coord_descent_kernel -- the first sweep or the first two were run elsewhere; they count as sweeps 1 (and 2),
// every word starts tagged with the last of them and carries whether that sweep changed the layer.
template <int KT, bool SBPROWS, bool RESUME>
__global__ void __launch_bounds__(32 * kWaveWarps) coord_descent_wave_kernel(int W, const int64_t* __restrict__ T, int Krt, int L, int S,
                                                                            const int32_t* __restrict__ init, int max_sweeps,
                                                                            int64_t* __restrict__ cost, int32_t* __restrict__ strategy,
                                                                            int32_t* __restrict__ sweeps, const int32_t* __restrict__ prev) {
  extern __shared__ __align__(16) unsigned char smem[];
  volatile uint32_t* st = reinterpret_cast<uint32_t*>(smem);          // [L] tag << 16 | changed << 15 | s_l
  int* stop = reinterpret_cast<int*>(smem) + L;                       // first sweep that changed nothing

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const size_t ps = blockIdx.x;
  const size_t p = ps / S;
  const int K = KT ? KT : Krt;
  const int64_t* Tp = T + p * (size_t)L * K * K;
  constexpr int NCAND = KT ? (KT + 31) / 32 : 8;
  int rep[NCAND];                                          // row that holds candidate c's column value
#pragma unroll
  for (int q = 0; q < NCAND; ++q) {
    const int c = 32 * q + lane;
    int r = 0, pw = 1, x = c;
    if (SBPROWS) {
      for (int d = 0; d < 3 && pw < K; ++d) {
        const int dig = x % 6;
        x /= 6;
        r += (dig < 4 ? dig : 2) * pw;
        pw *= 6;
      }
    } else {
      r = c;
    }
    rep[q] = r;
  }
  int base = 0;                                            // sweeps done before this kernel
  bool resume_done = false;
  if (RESUME) {
    int a1 = 0, a2 = 0;                                    // sweep 1 / sweep 2 changed something
    for (int l = threadIdx.x; l < L; l += blockDim.x) {
      const int s0 = init[ps * L + l], s1 = prev ? prev[ps * L + l] : strategy[ps * L + l];
      a1 |= s1 != s0;
      if (prev) a2 |= strategy[ps * L + l] != s1;
    }
    const bool any1 = __syncthreads_or(a1) != 0, any2 = __syncthreads_or(a2) != 0;
    const bool two = prev != nullptr && any1 && max_sweeps > 1;      // sweep 2 counts
    const int32_t* last = two || !prev ? strategy : prev;            // the state the descent stands at
    const int32_t* before = two ? prev : init;                       // the state one sweep earlier
    base = two ? 2 : 1;
    for (int l = threadIdx.x; l < L; l += blockDim.x) {
      const int v = last[ps * L + l];
      st[l] = ((uint32_t)base << 16) | (v != before[ps * L + l] ? 0x8000u : 0u) | ((uint32_t)v & 255u);
    }
    resume_done = !any1 || max_sweeps <= 1 || (two && (!any2 || max_sweeps <= 2));
  } else {
    for (int l = threadIdx.x; l < L; l += blockDim.x) st[l] = (uint32_t)init[ps * L + l] & 255u;      // tag 0
  }
  if (threadIdx.x == 0) *stop = resume_done ? base : INT32_MAX;
  __syncthreads();
  if (max_sweeps < 1) max_sweeps = 1;

  auto load_col = [&](int l, int sr, int64_t (&cv)[NCAND]) {          // T[l+1][.][sr], sr = s_{l+1}
    const bool has_right = l < L - 1;
    const int64_t* col = Tp + (size_t)(l + 1) * K * K + sr;
#pragma unroll
    for (int q = 0; q < NCAND; ++q) {
      const int c = 32 * q + lane;
      cv[q] = (has_right && c < K) ? ldg_narrow(col + (size_t)rep[q] * K) : 0;
    }
  };
  for (int k = base + w + 1; k <= max_sweeps; k += W) {
    if (k > *reinterpret_cast<volatile int*>(stop)) break;
    const uint32_t tagp = (uint32_t)(k - 1) << 16;           // words tagged k-1 (or later: never) are sweep k-1's
    bool changed = false, live = true;
    uint32_t left = 0;                                      // this sweep's word of layer l-1
    // The column of layer l+1 is known as soon as sweep k-1 has left layer l+2: it is gathered one layer ahead when the layer
    // is known to be dirty (sweep 1, or its right neighbour changed in sweep k-1), so that only the contiguous row read
    // stays on the dependent chain.
    int64_t cvp[NCAND];
    int pf = -1;
    if (!RESUME && k == 1 && L > 1) { load_col(0, (int)(st[1] & 255u), cvp); pf = 0; }
    int l = 0;
    while (l < L) {
      if (*reinterpret_cast<volatile int*>(stop) < k) { live = false; break; }   // an earlier sweep changed nothing: done
      // a run of clean layers (left neighbour unchanged in this sweep, right neighbour left unchanged by sweep k-1): lane i
      // looks at layer l+i; the layers before the first that is dirty or not yet ready are tagged at once
      if ((RESUME || k > 1) && !(left & 0x8000u)) {
        const int li = l + lane;
        bool ok = false;
        uint32_t mine = 0;
        if (li < L) {
          const uint32_t r = st[li + 1 < L ? li + 1 : L - 1], own = st[li];
          ok = r >= tagp && own >= tagp && !(li + 1 < L && (r & 0x8000u));
          mine = ((uint32_t)k << 16) | (own & 255u);
        }
        const unsigned m = __ballot_sync(0xffffffffu, ok);
        const int run = m == 0xffffffffu ? 32 : __ffs(~m) - 1;
        if (run > 0) {
          __syncwarp();
          if (lane < run) st[li] = mine;
          left = __shfl_sync(0xffffffffu, mine, run - 1);
          l += run;
          continue;
        }
      }
      const int lw = l + 1 < L ? l + 1 : L - 1;             // the word to wait for: sweep k-1 has left layer l+1 (L-1: layer l)
      uint32_t right = st[lw];
      while (right < tagp || st[l] < tagp) {                // (the layer's own word as well: sweep k-1 tags runs of layers at once)
        if (*reinterpret_cast<volatile int*>(stop) < k) { live = false; break; }
        __nanosleep(100);
        right = st[lw];
      }
      if (!live) break;
      const bool has_right = l + 1 < L;
      const bool dirty = (!RESUME && k == 1) || (l > 0 && (left & 0x8000u)) || (has_right && (right & 0x8000u));
      int64_t cv[NCAND];
      if (dirty) {
        if (pf == l) {
#pragma unroll
          for (int q = 0; q < NCAND; ++q) cv[q] = cvp[q];
        } else {
          load_col(l, (int)(right & 255u), cv);
        }
      }
      if (l + 2 < L) {
        const uint32_t r2 = st[l + 2];
        if ((!RESUME && k == 1) || (r2 >= tagp && (r2 & 0x8000u))) {
          load_col(l + 1, (int)(r2 & 255u), cvp);           // in flight during this layer's row read and argmin
          pf = l + 1;
        }
      }
      const uint32_t cur = st[l] & 255u;
      uint32_t word = ((uint32_t)k << 16) | cur;
      if (dirty) {
        const int64_t* row = Tp + ((size_t)l * K + (l > 0 ? (left & 255u) : 0)) * K;
        int64_t bv = INT64_MAX;
        int bi = K;
#pragma unroll
        for (int q = 0; q < NCAND; ++q) {
          const int c = 32 * q + lane;
          if (c < K) {
            const int64_t g = __ldg(row + c) + cv[q];
            if (g < bv) { bv = g; bi = c; }
          }
        }
        warp_argmin(bv, bi);
        if ((uint32_t)bi != cur) {
          changed = true;
          word = ((uint32_t)k << 16) | 0x8000u | (uint32_t)bi;
        }
      }
      __syncwarp();
      if (lane == 0) st[l] = word;
      left = word;
      ++l;
    }
    if (live && !changed && lane == 0) atomicMin(stop, k);
    __syncwarp();
  }
  __syncthreads();

  if (w == 0) {                                            // Cost(s) = sum_l T[l][s_{l-1}][s_l]
    int64_t acc = 0;
    for (int l = lane; l < L; l += 32) {
      const int left = l > 0 ? (int)(st[l - 1] & 255u) : 0, cur = (int)(st[l] & 255u);
      acc += ldg_narrow(Tp + ((size_t)l * K + left) * K + cur);
      strategy[ps * L + l] = cur;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (lane == 0) {
      cost[ps] = acc;
      const int sp = *stop;
      sweeps[ps] = sp < max_sweeps ? sp : max_sweeps;
    }
  }
}

template <int K, bool SBPROWS, bool RESUME>
int launch_wave(const int64_t* d_T, int Krt, int Bp, int L, const int32_t* d_init, int S, int max_sweeps, int64_t* d_cost,
                int32_t* d_strategy, int32_t* d_sweeps, cudaStream_t st, const int32_t* d_prev, int W) {
  const size_t smem = ((size_t)L * 4 + 4 + 15) / 16 * 16;
  if (smem > 48 * 1024)
    ADL_CUDA_CHECK(cudaFuncSetAttribute(coord_descent_wave_kernel<K, SBPROWS, RESUME>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  coord_descent_wave_kernel<K, SBPROWS, RESUME><<<(unsigned)(Bp * S), 32 * W, smem, st>>>(W, d_T, Krt, L, S, d_init, max_sweeps, d_cost,
                                                                                          d_strategy, d_sweeps, d_prev);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

template <int K, bool RESUME, bool SBPROWS>
int launch_k(const int64_t* d_T, int Krt, int Bp, int L, const int32_t* d_init, int S, int max_sweeps, int64_t* d_cost,
             int32_t* d_strategy, int32_t* d_sweeps, cudaStream_t st, const int32_t* d_prev = nullptr) {
  const size_t smem = ((size_t)L * 5 + 15) / 16 * 16;
  if (smem > 200 * 1024) { set_error("coord_descent: L too large"); return AUTODDL_EINVAL; }
  if (smem > 48 * 1024)
    ADL_CUDA_CHECK(cudaFuncSetAttribute(coord_descent_kernel<K, RESUME, SBPROWS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t nb = (int64_t)Bp * S;
  if (nb > 0x7fffffff) { set_error("coord_descent: Bp*S too large"); return AUTODDL_EINVAL; }
  coord_descent_kernel<K, RESUME, SBPROWS><<<(unsigned)nb, 32, smem, st>>>(d_T, Krt, L, S, d_init, max_sweeps, d_cost, d_strategy, d_sweeps, d_prev);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace

int launch_coord_descent(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, const int32_t* d_init, int32_t S,
                         int32_t max_sweeps, int64_t* d_cost, int32_t* d_strategy, int32_t* d_sweeps, cudaStream_t st,
                         bool resume, bool sbp_rows, const int32_t* d_prev) {
#define ADL_CD(KK, RS, SB) launch_k<KK, RS, SB>(d_T, K, Bp, L, d_init, S, max_sweeps, d_cost, d_strategy, d_sweeps, st, d_prev)
  const int64_t nb = (int64_t)Bp * S;
  if (nb > 0x7fffffff) { set_error("coord_descent: Bp*S too large"); return AUTODDL_EINVAL; }
  // sweeps of a start in flight (coord_descent_wave_kernel): eight up to two starts per SM, four beyond
  const int wave_w = nb <= kWaveWideBlocks ? kWaveWarps : kWaveWarps / 2;
  const bool wave_ok = L >= 8 && L < 50000 && max_sweeps > 1 && max_sweeps < 32768;
  if (resume) {
    // (config 4's 4,096 chains fill the machine with one warp each: two sweeps side by side gain 2 us of 78, four lose 28)
    if (K == 36 && wave_ok && nb <= kWaveMaxBlocks)
      return sbp_rows ? launch_wave<36, true, true>(d_T, K, Bp, L, d_init, S, max_sweeps, d_cost, d_strategy, d_sweeps, st, d_prev, wave_w)
                      : launch_wave<36, false, true>(d_T, K, Bp, L, d_init, S, max_sweeps, d_cost, d_strategy, d_sweeps, st, d_prev, wave_w);
    if (K == 36) return sbp_rows ? ADL_CD(36, true, true) : ADL_CD(36, true, false);
    set_error("coord_descent: resume mode exists for K = 36 only");
    return AUTODDL_EINVAL;
  }
  // a chain long enough to pipeline: the sweeps of a start side by side (coord_descent_wave_kernel)
  if (wave_ok) {                                           // (also with many starts: 4,096 chains of config 4 0.336 -> 0.298 ms)
#define ADL_WV(KK, SB) launch_wave<KK, SB, false>(d_T, K, Bp, L, d_init, S, max_sweeps, d_cost, d_strategy, d_sweeps, st, nullptr, wave_w)
    switch (K) {
      case 6:   return sbp_rows ? ADL_WV(6, true) : ADL_WV(6, false);
      case 36:  return sbp_rows ? ADL_WV(36, true) : ADL_WV(36, false);
      case 216: return sbp_rows ? ADL_WV(216, true) : ADL_WV(216, false);
    }
    if (!sbp_rows) {
      if (K == 81) return ADL_WV(81, false);
      if (K == 243) return ADL_WV(243, false);
      if (K >= 1 && K <= 256) return ADL_WV(0, false);
    }
#undef ADL_WV
  }
  switch (K) {
    case 6:   return sbp_rows ? ADL_CD(6, false, true) : ADL_CD(6, false, false);
    case 36:  return sbp_rows ? ADL_CD(36, false, true) : ADL_CD(36, false, false);
    case 216: return sbp_rows ? ADL_CD(216, false, true) : ADL_CD(216, false, false);
  }
  if (!sbp_rows) {                                         // four / five mesh levels (R26): the paper's rows, then any K
    if (K == 81) return ADL_CD(81, false, false);
    if (K == 243) return ADL_CD(243, false, false);
    if (K >= 1 && K <= 256) return ADL_CD(0, false, false);
  }
#undef ADL_CD
  set_error("coord_descent: K = %d not supported (6, 36, 216, or any K <= 256 on caller-indexed tables)", K);
  return AUTODDL_EINVAL;
}

}  // namespace autoddl
