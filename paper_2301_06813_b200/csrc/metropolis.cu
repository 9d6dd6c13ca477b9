// Metropolis-Hastings sampler over the cost tables (R19-R22) for sm_100a.
//
// P(S) ~ exp(-Cost(S) / tau).  Step t of a chain proposes s_l <- s' for one layer l and accepts with probability
// min(1, P(S_new) / P(S_old)) = min(1, exp(-dC / tau)); dC touches four table cells.  The draws (l, s', u) of
// step t come from a counter-based generator (the n-th output of splitmix64), so they are known in advance.
//
// One warp per chain; the chain itself is sequential, but its proposals are not: lane k of the warp evaluates
// step t + k against the state at the start of the window (two scattered 8-byte loads per lane for the proposed
// cells, all 64 in flight at once; the two cells of the current state come from a per-layer cache
// e[l] = T[l][s_{l-1}][s_l] in shared memory, which a committed move refreshes from the cells it has just read), then
// the warp commits the steps in order: a step stays valid as long as no earlier step of the window changed a layer
// within distance 1 of its own; the window is cut at the first invalidated step, which is
// re-evaluated in the next round.  The committed trajectory is exactly the sequential one.
//
// The acceptance test is integer only (bit-exact against the oracle): accept iff dC <= 0 or
//   dC < 2^45  and  tau * neglog_q16(x) >= dC * 2^16,   x = (u >> 32) + 1 in [1, 2^32],
// neglog_q16(x) = -ln(x / 2^32) in Q16 by sixteen shift-and-square steps on a Q62 mantissa.
#include "common.cuh"

namespace autoddl {

namespace {

__device__ __forceinline__ uint64_t splitmix_nth(uint64_t seed, uint64_t n) {
  uint64_t z = seed + n * 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// -ln(x / 2^32) * 2^16 for x in [1, 2^32]; every product truncated to Q62 (R21)
__device__ __forceinline__ int64_t neglog_q16(uint64_t x) {
  const int n = 63 - __clzll((long long)x);
  uint64_t m = x << (62 - n);                              // Q62 in [2^62, 2^63)
  uint32_t frac = 0;
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const uint64_t hi = __umul64hi(m, m), lo = m * m;      // Q124
    m = (hi << 2) | (lo >> 62);                            // Q62 in [2^62, 2^64)
    frac <<= 1;
    if (m >> 63) { frac |= 1; m >>= 1; }
  }
  const int64_t log2_q16 = ((int64_t)n << 16) | (int64_t)frac;
  const int64_t nlog2_q16 = ((int64_t)32 << 16) - log2_q16;
  return (nlog2_q16 * 744261117ll) >> 30;                  // ln 2 = 744261117 / 2^30, truncated
}

// x mod d for any 64-bit x with the launch constant M = floor(2^64 / d): the multiply-high quotient is short by at most
// two, so two conditional subtractions make the remainder exact (a run-time 64-bit division costs ~5x as much)
__device__ __forceinline__ uint32_t mod_magic(uint64_t x, uint32_t d, uint64_t M) {
  uint64_t r = x - __umul64hi(x, M) * d;
  if (r >= d) r -= d;
  if (r >= d) r -= d;
  return (uint32_t)r;
}

__device__ __forceinline__ int64_t ldg64(const int64_t* p) {
  int64_t v;
  asm volatile("ld.global.nc.L2::64B.b64 %0, [%1];" : "=l"(v) : "l"(p));
  return v;
}

constexpr int kWarps = 4;                                  // chains per block

__global__ void __launch_bounds__(kWarps * 32)
metropolis_kernel(const int64_t* __restrict__ T, int nchains, int L, int K, int S, const int32_t* __restrict__ init,
                  int nsteps, int64_t tau, uint64_t seed, uint64_t magicL, uint64_t magicK, int64_t* __restrict__ best_cost,
                  int32_t* __restrict__ best_strategy, int64_t* __restrict__ final_cost,
                  int32_t* __restrict__ final_strategy, int32_t* __restrict__ accepted) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int64_t chain = (int64_t)blockIdx.x * kWarps + wib;
  if (chain >= nchains) return;
  int64_t* e = reinterpret_cast<int64_t*>(smem) + (size_t)wib * L;          // e[l] = T[l][s_{l-1}][s_l] of the current state
  uint8_t* s = smem + (size_t)kWarps * L * 8 + (size_t)wib * 2 * L;         // current strategy [L]
  uint8_t* sb = s + L;                                     // best strategy [L]
  const int64_t* Tp = T + (chain / S) * (int64_t)L * K * K;

  // start: s = init, cur = Cost(init)
  int64_t part = 0;
  for (int l = lane; l < L; l += 32) {
    const int v = init[chain * L + l];
    s[l] = (uint8_t)v;
    sb[l] = (uint8_t)v;
  }
  __syncwarp();
  for (int l = lane; l < L; l += 32) {
    e[l] = ldg64(Tp + ((int64_t)l * K + (l > 0 ? s[l - 1] : 0)) * K + s[l]);
    part += e[l];
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) part += __shfl_xor_sync(0xffffffffu, part, off);
  int64_t cur = part, best = part;
  int nacc = 0;

  int t = 0;
  while (t < nsteps) {
    // ---- evaluate steps t .. t+31 against the current state -------------------------------------------------
    const int tk = t + lane;
    const bool live = tk < nsteps;
    const uint64_t base = (((uint64_t)chain << 32) + (uint64_t)(live ? tk : 0)) * 4;
    const int l = (int)mod_magic(splitmix_nth(seed, base + 1), (uint32_t)L, magicL);
    const int c = (int)mod_magic(splitmix_nth(seed, base + 2), (uint32_t)K, magicK);
    const uint64_t x = (splitmix_nth(seed, base + 3) >> 32) + 1;
    const int old = s[l];
    const int left = l > 0 ? s[l - 1] : 0;
    const int64_t n0 = ldg64(Tp + ((int64_t)l * K + left) * K + c);                       // T[l][s_{l-1}][s']
    const int64_t n1 = l < L - 1 ? ldg64(Tp + ((int64_t)(l + 1) * K + c) * K + s[l + 1]) : 0;   // T[l+1][s'][s_{l+1}]
    int64_t d = n0 - e[l];
    if (l < L - 1) d += n1 - e[l + 1];
    bool acc = d <= 0;
    if (!acc && d < ((int64_t)1 << 45)) acc = tau * neglog_q16(x) >= (d << 16);
    acc = acc && live;
    const bool chg = acc && c != old;

    // ---- commit in order ---------------------------------------------------------------------------------------
    const unsigned live_mask = __ballot_sync(0xffffffffu, live);
    const unsigned acc_mask = __ballot_sync(0xffffffffu, acc);
    unsigned chg_mask = __ballot_sync(0xffffffffu, chg);
    int end = __popc(live_mask);                           // steps of this window that are committed: [0, end)
    while (chg_mask) {
      const int j = __ffs(chg_mask) - 1;
      if (j >= end) break;
      const int lj = __shfl_sync(0xffffffffu, l, j);
      const int cj = __shfl_sync(0xffffffffu, c, j);
      const int64_t dj = __shfl_sync(0xffffffffu, d, j);
      const int64_t n0j = __shfl_sync(0xffffffffu, n0, j), n1j = __shfl_sync(0xffffffffu, n1, j);
      cur += dj;
      if (lane == 0) {
        s[lj] = (uint8_t)cj;
        e[lj] = n0j;
        if (lj < L - 1) e[lj + 1] = n1j;
      }
      __syncwarp();
      if (cur < best) {                                     // first time this cost is attained
        best = cur;
        for (int q = lane; q < L; q += 32) sb[q] = s[q];
      }
      // later steps that read a layer within distance 1 of lj must be evaluated again
      const int dist = l - lj;
      const unsigned inval = __ballot_sync(0xffffffffu, dist >= -1 && dist <= 1) & ~((2u << j) - 1u);
      if (inval) {
        const int lim = __ffs(inval) - 1;
        if (lim < end) end = lim;
      }
      chg_mask &= ~((2u << j) - 1u);
    }
    nacc += __popc(acc_mask & (end >= 32 ? 0xffffffffu : ((1u << end) - 1u)));
    t += end;
    __syncwarp();
  }

  if (lane == 0) {
    best_cost[chain] = best;
    final_cost[chain] = cur;
    accepted[chain] = nacc;
  }
  for (int l = lane; l < L; l += 32) {
    best_strategy[chain * L + l] = sb[l];
    final_strategy[chain * L + l] = s[l];
  }
}

}  // namespace

int launch_metropolis(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, const int32_t* d_init, int32_t S,
                      int32_t nsteps, int64_t tau_ps, uint64_t seed, int64_t* d_best_cost, int32_t* d_best_strategy,
                      int64_t* d_final_cost, int32_t* d_final_strategy, int32_t* d_accepted, cudaStream_t st) {
  const int64_t nchains = (int64_t)Bp * S;
  if (nchains > 0x3fffffff) { set_error("metropolis: Bp*S too large"); return AUTODDL_EINVAL; }
  if (K > 256) { set_error("metropolis: K must be <= 256"); return AUTODDL_EINVAL; }
  const size_t smem = ((size_t)kWarps * (8 + 2) * L + 15) / 16 * 16;
  if (smem > 200 * 1024) { set_error("metropolis: L too large"); return AUTODDL_EINVAL; }
  if (smem > 48 * 1024)
    ADL_CUDA_CHECK(cudaFuncSetAttribute(metropolis_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const unsigned grid = (unsigned)((nchains + kWarps - 1) / kWarps);
  // floor(2^64 / d); d = 1 would need 2^64: every x mod 1 is 0, which M = 0 also yields (r = x, two subtractions of 1 are
  // not enough), so d = 1 uses M = 2^64 - 1: quotient x - 1 for x >= 1, remainder 1 -> corrected to 0
  auto magic = [](uint32_t d) { return d == 1 ? ~(uint64_t)0 : (uint64_t)((((unsigned __int128)1) << 64) / d); };
  metropolis_kernel<<<grid, kWarps * 32, smem, st>>>(d_T, (int)nchains, L, K, S, d_init, nsteps, tau_ps, seed,
                                                     magic((uint32_t)L), magic((uint32_t)K), d_best_cost,
                                                     d_best_strategy, d_final_cost, d_final_strategy, d_accepted);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
