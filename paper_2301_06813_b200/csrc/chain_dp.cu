// (a2) Exact min-plus chain DP for sm_100a.  DESIGN.md R9; the optimum equals the paper's exhaustive
// search.
//
//   f_0[j] = T[0][0][j];  f_l[j] = min_i f_{l-1}[i] + T[l][i][j]  (smallest i on ties);  backtrack.
//
// One CTA per problem.  A producer warp streams the problem's tiles through a ring of shared-memory
// stages with TMA bulk copies (cp.async.bulk + mbarrier complete_tx, L2 evict-first: every byte is read
// once).  Consumer threads each own a pair of adjacent columns (one 16-byte shared load per row) and a
// group of rows; f is broadcast from shared memory.  With one consumer warp (K = 36) a layer needs no
// block barrier at all; with several row groups (K = 216) partial minima are merged through shared
// memory with the lexicographic (value, row) order that keeps the lowest-index tie-break.

#include "common.cuh"

namespace autoddl {

namespace {

struct DpCfg {
  int K;        // signatures
  int RB;       // rows per stage
  int STAGES;
  int G;        // row groups (consumer threads = G * K/2, rounded up to warps)
};

template <int K, int RB, int STAGES, int G>
struct DpLayout {
  static constexpr int KH = K / 2;
  static constexpr int NCONS = ((G * KH + 31) / 32) * 32;   // consumer threads
  static constexpr int NT = NCONS + 32;                     // + producer warp
  static constexpr int STAGE_BYTES = RB * K * 8;
  static constexpr int NBLK = K / RB;                       // row blocks per tile
  static_assert(K % RB == 0, "RB must divide K");
  static_assert(RB % G == 0, "G must divide RB");
  static_assert(STAGE_BYTES % 16 == 0, "bulk copy granularity");
};

__device__ __forceinline__ bool lex_less(int64_t v, int i, int64_t bv, int bi) {
  return v < bv || (v == bv && i < bi);
}

template <int K, int RB, int STAGES, int G, bool BP_SMEM>
__global__ void __launch_bounds__(DpLayout<K, RB, STAGES, G>::NT)
chain_dp_kernel(const int64_t* __restrict__ T, int L, uint8_t* __restrict__ bp_glob,
                int64_t* __restrict__ opt_cost, int32_t* __restrict__ strategy) {
  using Lay = DpLayout<K, RB, STAGES, G>;
  constexpr int KH = Lay::KH, NCONS = Lay::NCONS, NBLK = Lay::NBLK, SB = Lay::STAGE_BYTES;
  constexpr int RPG = RB / G;                                // rows per group per stage

  extern __shared__ __align__(128) unsigned char smem[];
  // layout: stages | f[2][K] | part (G>1) | full[STAGES] empty[STAGES] | bp (optional) | strat
  int64_t* stage0 = reinterpret_cast<int64_t*>(smem);
  int64_t* fbuf = reinterpret_cast<int64_t*>(smem + (size_t)STAGES * SB);
  int64_t* partv = fbuf + 2 * K;                             // [G][K] values
  int32_t* parti = reinterpret_cast<int32_t*>(partv + (G > 1 ? G * K : 0));   // [G][K] rows
  uint64_t* full = reinterpret_cast<uint64_t*>(parti + (G > 1 ? G * K : 0) + ((G > 1 ? G * K : 0) & 1));
  uint64_t* empty = full + STAGES;
  uint8_t* bp_s = reinterpret_cast<uint8_t*>(empty + STAGES);

  const int tid = threadIdx.x;
  const int p = blockIdx.x;
  const int64_t* Tp = T + (size_t)p * L * K * K;
  uint8_t* bp = BP_SMEM ? bp_s : bp_glob + (size_t)p * L * K;

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], NCONS / 32);                      // one arrive per consumer warp
    }
    mbar_fence_init();
  }
  __syncthreads();

  const int nblocks = (L - 1) * NBLK;                        // tile 0 contributes only its row 0

  if (tid >= NCONS) {
    // ================= producer warp: one elected lane drives TMA =================
    if (tid == NCONS) {
      const uint64_t pol = policy_evict_first();
      const unsigned char* src = reinterpret_cast<const unsigned char*>(Tp + (size_t)K * K);
      for (int b = 0; b < nblocks; ++b) {
        const int s = b % STAGES;
        if (b >= STAGES) mbar_wait(&empty[s], ((b / STAGES) - 1) & 1);
        mbar_arrive_expect_tx(&full[s], SB);
        bulk_g2s(smem + (size_t)s * SB, src + (size_t)b * SB, SB, &full[s], pol);
      }
    }
    return;
  }

  // ================= consumers =================
  const int cp = tid % KH;                                   // column pair
  const int g = tid / KH;                                    // row group (>= G: idle padding lanes)
  const bool active = g < G;
  const int lane = tid & 31;

  // f_0 = row 0 of tile 0
  for (int j = tid; j < K; j += NCONS) fbuf[j] = __ldg(Tp + j);
  if (G > 1 || NCONS > 32) asm volatile("bar.sync 1, %0;" ::"n"(NCONS)); else __syncwarp();

  int cur = 0;
  int b = 0;
  for (int l = 1; l < L; ++l) {
    const int64_t* f = fbuf + cur * K;
    int64_t best0 = INT64_MAX, best1 = INT64_MAX;     // cells < 2^62/L: the first row always wins
    int a0 = 0, a1 = 0;
    for (int rb = 0; rb < NBLK; ++rb, ++b) {
      const int s = b % STAGES;
      mbar_wait(&full[s], (b / STAGES) & 1);
      if (active) {
        const int64_t* tile = stage0 + (size_t)s * (SB / 8);
#pragma unroll 6
        for (int r = 0; r < RPG; ++r) {
          const int rl = g * RPG + r;                        // row inside the stage
          const int i = rb * RB + rl;
          const int64_t fi = f[i];
          const longlong2 t = *reinterpret_cast<const longlong2*>(tile + rl * K + 2 * cp);
          const int64_t v0 = fi + t.x, v1 = fi + t.y;
          if (v0 < best0) { best0 = v0; a0 = i; }
          if (v1 < best1) { best1 = v1; a1 = i; }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);                 // this warp is done with the stage
    }
    int64_t* fn = fbuf + (cur ^ 1) * K;
    if (G == 1) {
      if (active) {
        *reinterpret_cast<longlong2*>(fn + 2 * cp) = make_longlong2(best0, best1);
        bp[(size_t)l * K + 2 * cp] = (uint8_t)a0;
        bp[(size_t)l * K + 2 * cp + 1] = (uint8_t)a1;
      }
      if (NCONS > 32) asm volatile("bar.sync 1, %0;" ::"n"(NCONS)); else __syncwarp();
    } else {
      if (active) {
        partv[g * K + 2 * cp] = best0;  parti[g * K + 2 * cp] = a0;
        partv[g * K + 2 * cp + 1] = best1;  parti[g * K + 2 * cp + 1] = a1;
      }
      asm volatile("bar.sync 1, %0;" ::"n"(NCONS));
      for (int j = tid; j < K; j += NCONS) {
        int64_t bv = partv[j];
        int bi = parti[j];
#pragma unroll
        for (int gg = 1; gg < G; ++gg) {
          const int64_t v = partv[gg * K + j];
          const int i = parti[gg * K + j];
          if (lex_less(v, i, bv, bi)) { bv = v; bi = i; }
        }
        fn[j] = bv;
        bp[(size_t)l * K + j] = (uint8_t)bi;
      }
      asm volatile("bar.sync 1, %0;" ::"n"(NCONS));
    }
    cur ^= 1;
  }

  // ---- smallest argmin of f_{L-1}, backtrack -------------------------------------------------------
  if (tid < 32) {
    const int64_t* f = fbuf + cur * K;
    int64_t bv = 0;
    int bi = -1;
    for (int j = lane; j < K; j += 32) {
      const int64_t v = f[j];
      if (bi < 0 || v < bv) { bv = v; bi = j; }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (oi >= 0 && (bi < 0 || lex_less(ov, oi, bv, bi))) { bv = ov; bi = oi; }
    }
    int32_t* sp = strategy + (size_t)p * L;
    if (lane == 0) {
      opt_cost[p] = bv;
      int s = bi;
      sp[L - 1] = s;
      for (int l = L - 1; l >= 1; --l) {
        s = bp[(size_t)l * K + s];
        sp[l - 1] = s;
      }
    }
  }
}

// ---- K = 36 (two mesh levels): one consumer warp with all 32 lanes busy --------------------------------
// Columns 0..31: lane = h*16 + c owns columns (2c, 2c+1) and rows [18h, 18h+18): one 16-byte shared load per
// row, the two halves merged with one shuffle step.  Columns 32..35: lane = g*4 + cc owns column 32+cc and
// rows g, g+8, ..., merged over the 8 row groups with three shuffle steps.  Every merge compares
// (value, row) lexicographically, so the smallest row wins ties exactly as in the sequential definition.
template <int STAGES>
__global__ void __launch_bounds__(64)
chain_dp36_kernel(const int64_t* __restrict__ T, int L, int64_t* __restrict__ opt_cost, int32_t* __restrict__ strategy) {
  constexpr int K = 36, SB = K * K * 8;
  extern __shared__ __align__(128) unsigned char smem[];
  int64_t* stage0 = reinterpret_cast<int64_t*>(smem);
  int64_t* fbuf = reinterpret_cast<int64_t*>(smem + (size_t)STAGES * SB);      // [2][K]
  uint64_t* full = reinterpret_cast<uint64_t*>(fbuf + 2 * K);
  uint64_t* empty = full + STAGES;
  uint8_t* bp = reinterpret_cast<uint8_t*>(empty + STAGES);                     // [L][K]

  const int tid = threadIdx.x;
  const int p = blockIdx.x;
  const int64_t* Tp = T + (size_t)p * L * K * K;

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    mbar_fence_init();
  }
  __syncthreads();

  if (tid >= 32) {                         // producer warp: one lane drives the TMA ring
    if (tid == 32) {
      const uint64_t pol = policy_evict_first();
      const unsigned char* src = reinterpret_cast<const unsigned char*>(Tp + (size_t)K * K);
      for (int b = 0; b < L - 1; ++b) {
        const int s = b % STAGES;
        if (b >= STAGES) mbar_wait(&empty[s], ((b / STAGES) - 1) & 1);
        mbar_arrive_expect_tx(&full[s], SB);
        bulk_g2s(smem + (size_t)s * SB, src + (size_t)b * SB, SB, &full[s], pol);
      }
    }
    return;
  }

  const int lane = tid;
  const int c = lane & 15, h = lane >> 4;          // main part
  const int cc = lane & 3, g = lane >> 2;          // remainder part
  for (int j = lane; j < K; j += 32) fbuf[j] = __ldg(Tp + j);     // f_0 = row 0 of tile 0
  __syncwarp();

  int cur = 0;
  for (int l = 1; l < L; ++l) {
    const int b = l - 1, s = b % STAGES;
    const int64_t* f = fbuf + cur * K;
    const int64_t* tile = stage0 + (size_t)s * (SB / 8);
    mbar_wait(&full[s], (b / STAGES) & 1);

    int64_t best0, best1, bestr = INT64_MAX;
    int a0, a1, ar = 0;
    const int64_t* trow = tile + (18 * h) * K + 2 * c;
    const int64_t* frow = f + 18 * h;
    {
      // three independent chains of six rows per column (instruction-level parallelism; one exposed chain of 18 is what
      // a single long problem waits for), merged in row order: strict '<' keeps the smallest index
      int64_t p0[3], p1[3];
      int q0[3], q1[3];
#pragma unroll
      for (int part = 0; part < 3; ++part) {
        longlong2 t[6];
        int64_t fi[6];
#pragma unroll
        for (int r = 0; r < 6; ++r) {
          t[r] = *reinterpret_cast<const longlong2*>(trow + (6 * part + r) * K);
          fi[r] = frow[6 * part + r];
        }
        int64_t b0 = fi[0] + t[0].x, b1 = fi[0] + t[0].y;
        int i0 = 6 * part, i1 = 6 * part;
#pragma unroll
        for (int r = 1; r < 6; ++r) {
          const int64_t v0 = fi[r] + t[r].x, v1 = fi[r] + t[r].y;
          if (v0 < b0) { b0 = v0; i0 = 6 * part + r; }
          if (v1 < b1) { b1 = v1; i1 = 6 * part + r; }
        }
        p0[part] = b0; q0[part] = i0; p1[part] = b1; q1[part] = i1;
      }
      best0 = p0[0]; a0 = q0[0]; best1 = p1[0]; a1 = q1[0];
      if (p0[1] < best0) { best0 = p0[1]; a0 = q0[1]; }
      if (p0[2] < best0) { best0 = p0[2]; a0 = q0[2]; }
      if (p1[1] < best1) { best1 = p1[1]; a1 = q1[1]; }
      if (p1[2] < best1) { best1 = p1[2]; a1 = q1[2]; }
      a0 += 18 * h;
      a1 += 18 * h;
    }
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const int i = g + 8 * k;
      if (i < K) {
        const int64_t v = f[i] + tile[i * K + 32 + cc];
        if (v < bestr) { bestr = v; ar = i; }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);           // stage consumed: the producer may refill it

    {                                                // merge the two row halves
      const int64_t o0 = __shfl_xor_sync(0xffffffffu, best0, 16), o1 = __shfl_xor_sync(0xffffffffu, best1, 16);
      const int q0 = __shfl_xor_sync(0xffffffffu, a0, 16), q1 = __shfl_xor_sync(0xffffffffu, a1, 16);
      if (lex_less(o0, q0, best0, a0)) { best0 = o0; a0 = q0; }
      if (lex_less(o1, q1, best1, a1)) { best1 = o1; a1 = q1; }
    }
#pragma unroll
    for (int off = 4; off <= 16; off <<= 1) {        // merge the eight row groups
      const int64_t o = __shfl_xor_sync(0xffffffffu, bestr, off);
      const int q = __shfl_xor_sync(0xffffffffu, ar, off);
      if (lex_less(o, q, bestr, ar)) { bestr = o; ar = q; }
    }
    int64_t* fn = fbuf + (cur ^ 1) * K;
    uint8_t* bpl = bp + (size_t)l * K;
    if (lane < 16) {
      *reinterpret_cast<longlong2*>(fn + 2 * c) = make_longlong2(best0, best1);
      *reinterpret_cast<uint16_t*>(bpl + 2 * c) = (uint16_t)(a0 | a1 << 8);
    }
    if (lane < 4) {
      fn[32 + cc] = bestr;
      bpl[32 + cc] = (uint8_t)ar;
    }
    __syncwarp();
    cur ^= 1;
  }

  // smallest argmin of f_{L-1}, then backtrack
  const int64_t* f = fbuf + cur * K;
  int64_t bv = f[lane];
  int bi = lane;
  if (lane < K - 32) {
    const int64_t v = f[32 + lane];
    if (v < bv) { bv = v; bi = 32 + lane; }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
    if (lex_less(ov, oi, bv, bi)) { bv = ov; bi = oi; }
  }
  int32_t* sp = strategy + (size_t)p * L;
  if (lane == 0) {
    opt_cost[p] = bv;
    int sidx = bi;
    sp[L - 1] = sidx;
    for (int l = L - 1; l >= 1; --l) {
      sidx = bp[(size_t)l * K + sidx];
      sp[l - 1] = sidx;
    }
  }
}

template <int STAGES>
int launch_dp36(const int64_t* d_T, int Bp, int L, int64_t* d_opt, int32_t* d_strat, cudaStream_t st) {
  const size_t smem = ((size_t)STAGES * 36 * 36 * 8 + 2 * 36 * 8 + 2 * STAGES * 8 + (size_t)L * 36 + 127) / 128 * 128;
  auto kern = chain_dp36_kernel<STAGES>;
  ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<Bp, 64, smem, st>>>(d_T, L, d_opt, d_strat);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

template <int K, int RB, int STAGES, int G>
size_t dp_smem_bytes(int L, bool bp_smem) {
  using Lay = DpLayout<K, RB, STAGES, G>;
  size_t b = (size_t)STAGES * Lay::STAGE_BYTES + 2 * K * 8;
  if (G > 1) b += (size_t)G * K * 8 + (size_t)G * K * 4 + 8;
  b += 2 * STAGES * 8;
  if (bp_smem) b += (size_t)L * K;
  return (b + 127) / 128 * 128;
}

template <int K, int RB, int STAGES, int G>
int launch_cfg(const int64_t* d_T, int Bp, int L, uint8_t* d_bp, int64_t* d_opt, int32_t* d_strat, cudaStream_t st) {
  using Lay = DpLayout<K, RB, STAGES, G>;
  const bool bp_smem = (size_t)L * K <= 16 * 1024;
  if (!bp_smem && d_bp == nullptr) { set_error("chain_dp: workspace for back-pointers missing"); return AUTODDL_EWORK; }
  const size_t smem = dp_smem_bytes<K, RB, STAGES, G>(L, bp_smem);
  if (smem > 227 * 1024) { set_error("chain_dp: %zu bytes of shared memory needed", smem); return AUTODDL_EINVAL; }
  if (bp_smem) {
    auto kern = chain_dp_kernel<K, RB, STAGES, G, true>;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<Bp, Lay::NT, smem, st>>>(d_T, L, d_bp, d_opt, d_strat);
  } else {
    auto kern = chain_dp_kernel<K, RB, STAGES, G, false>;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<Bp, Lay::NT, smem, st>>>(d_T, L, d_bp, d_opt, d_strat);
  }
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

// ---- any K <= 256 (four / five mesh levels, R26: K = 81, 243, ... is odd, so neither the 16-byte column pairs nor
// the 16-byte-aligned TMA row blocks of the kernels above apply).  One CTA of 1024 threads per problem: thread
// (g, j) owns column j and the rows i = g, g + 4, ...; its loads do not depend on f, so eight of them are in flight
// per thread (8-byte loads, coalesced over j); the four row groups are merged through shared memory in the
// lexicographic (value, row) order.  Back-pointers live in shared memory when L * K fits, else in the workspace.
constexpr int kAnyG = 4, kAnyCols = 256;

// KT = 81, 243 (the paper's rows on four / five levels): K at compile time, row offsets become immediates; KT = 0: any K
template <int KT, bool BP_SMEM>
__global__ void __launch_bounds__(kAnyG * kAnyCols)
chain_dp_anyk_kernel(const int64_t* __restrict__ T, int L, int Krt, uint8_t* __restrict__ bp_glob,
                     int64_t* __restrict__ opt_cost, int32_t* __restrict__ strategy) {
  const int K = KT ? KT : Krt;
  extern __shared__ __align__(16) unsigned char smem[];
  int64_t* fbuf = reinterpret_cast<int64_t*>(smem);                  // [2][256]
  int64_t* partv = fbuf + 2 * kAnyCols;                              // [G][256]
  int32_t* parti = reinterpret_cast<int32_t*>(partv + kAnyG * kAnyCols);
  uint8_t* bp_s = reinterpret_cast<uint8_t*>(parti + kAnyG * kAnyCols);
  const int tid = threadIdx.x, j = tid % kAnyCols, g = tid / kAnyCols;
  const int p = blockIdx.x;
  const int64_t* Tp = T + (size_t)p * L * K * K;
  uint8_t* bp = BP_SMEM ? bp_s : bp_glob + (size_t)p * L * K;
  const bool active = j < K;

  if (g == 0 && active) fbuf[j] = __ldg(Tp + j);                     // f_0 = row 0 of tile 0
  __syncthreads();
  int cur = 0;
  for (int l = 1; l < L; ++l) {
    const int64_t* f = fbuf + cur * kAnyCols;
    const int64_t* tile = Tp + (size_t)l * K * K + j;
    int64_t best = INT64_MAX;
    int arg = 0;
    if (active) {
      int i = g;
      for (; i + 7 * kAnyG < K; i += 8 * kAnyG) {
        int64_t t[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) t[u] = __ldcs(tile + (size_t)(i + u * kAnyG) * K);
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const int64_t v = f[i + u * kAnyG] + t[u];
          if (v < best) { best = v; arg = i + u * kAnyG; }
        }
      }
      for (; i < K; i += kAnyG) {
        const int64_t v = f[i] + __ldcs(tile + (size_t)i * K);
        if (v < best) { best = v; arg = i; }
      }
      partv[g * kAnyCols + j] = best;
      parti[g * kAnyCols + j] = arg;
    }
    __syncthreads();
    if (g == 0 && active) {
      int64_t bv = partv[j];
      int bi = parti[j];
#pragma unroll
      for (int gg = 1; gg < kAnyG; ++gg) {
        const int64_t v = partv[gg * kAnyCols + j];
        const int i = parti[gg * kAnyCols + j];
        if (v != INT64_MAX && lex_less(v, i, bv, bi)) { bv = v; bi = i; }     // a group with no row (K < 4) holds no candidate
      }
      fbuf[(cur ^ 1) * kAnyCols + j] = bv;
      bp[(size_t)l * K + j] = (uint8_t)bi;
    }
    __syncthreads();
    cur ^= 1;
  }

  if (tid < 32) {                                                    // smallest argmin of f_{L-1}, backtrack
    const int lane = tid;
    const int64_t* f = fbuf + cur * kAnyCols;
    int64_t bv = 0;
    int bi = -1;
    for (int c = lane; c < K; c += 32) {
      const int64_t v = f[c];
      if (bi < 0 || v < bv) { bv = v; bi = c; }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (oi >= 0 && (bi < 0 || lex_less(ov, oi, bv, bi))) { bv = ov; bi = oi; }
    }
    int32_t* sp = strategy + (size_t)p * L;
    if (lane == 0) {
      opt_cost[p] = bv;
      int s = bi;
      sp[L - 1] = s;
      for (int l = L - 1; l >= 1; --l) {
        s = bp[(size_t)l * K + s];
        sp[l - 1] = s;
      }
    }
  }
}

int launch_anyk(const int64_t* d_T, int Bp, int L, int K, uint8_t* d_bp, int64_t* d_opt, int32_t* d_strat, cudaStream_t st) {
  const size_t base = (size_t)2 * kAnyCols * 8 + (size_t)kAnyG * kAnyCols * 12;
  const bool bp_smem = (size_t)L * K <= 16 * 1024;                  // same rule as the workspace sizing (api.cu)
  if (!bp_smem && d_bp == nullptr) { set_error("chain_dp: workspace for back-pointers missing"); return AUTODDL_EWORK; }
  const size_t smem = (base + (bp_smem ? (size_t)L * K : 0) + 127) / 128 * 128;
  if (bp_smem) {
    auto kern = K == 243 ? chain_dp_anyk_kernel<243, true> : K == 81 ? chain_dp_anyk_kernel<81, true> : chain_dp_anyk_kernel<0, true>;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<Bp, kAnyG * kAnyCols, smem, st>>>(d_T, L, K, d_bp, d_opt, d_strat);
  } else {
    auto kern = K == 243 ? chain_dp_anyk_kernel<243, false> : K == 81 ? chain_dp_anyk_kernel<81, false> : chain_dp_anyk_kernel<0, false>;
    kern<<<Bp, kAnyG * kAnyCols, smem, st>>>(d_T, L, K, d_bp, d_opt, d_strat);
  }
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace

int launch_chain_dp(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, uint8_t* d_bp, int64_t* d_opt_cost,
                    int32_t* d_strategy, cudaStream_t st) {
  switch (K) {
    case 6:   return launch_cfg<6, 6, 4, 1>(d_T, Bp, L, d_bp, d_opt_cost, d_strategy, st);
    case 36:
      if ((size_t)L * K <= 16 * 1024) {               // back-pointers fit in shared memory: the 32-lane kernel
        static const int stages = ADL_DEBUG_ENV_INT("AUTODDL_DP_STAGES", 3);
        if (stages == 2) return launch_dp36<2>(d_T, Bp, L, d_opt_cost, d_strategy, st);
        if (stages == 4) return launch_dp36<4>(d_T, Bp, L, d_opt_cost, d_strategy, st);
        return launch_dp36<3>(d_T, Bp, L, d_opt_cost, d_strategy, st);
      }
      return launch_cfg<36, 36, 3, 1>(d_T, Bp, L, d_bp, d_opt_cost, d_strategy, st);
    case 216: {
      // few long chains: one 8-CTA cluster per chain (chain_dp_cluster.cu); many chains already fill the machine
      static const bool no_cluster = ADL_DEBUG_ENV("AUTODDL_DP_NO_CLUSTER");
      if (!no_cluster && Bp * 8 <= device_sm_count() && chain_dp_cluster_supported(K, L)) {
        const int rc = launch_chain_dp_cluster(d_T, Bp, L, d_opt_cost, d_strategy, st);
        if (rc == AUTODDL_OK) return rc;
        cudaGetLastError();                                  // launch refused: fall back to one CTA per chain
        clear_error();
      }
      return launch_cfg<216, 24, 4, 8>(d_T, Bp, L, d_bp, d_opt_cost, d_strategy, st);
    }
  }
  if (K >= 1 && K <= 256) {
    static const bool no_cluster = ADL_DEBUG_ENV("AUTODDL_DP_NO_CLUSTER");
    if (!no_cluster && Bp * 8 <= device_sm_count() && chain_dp_cluster_anyk_supported(K, L)) {
      const int rc = launch_chain_dp_cluster_anyk(d_T, Bp, L, K, d_opt_cost, d_strategy, st);
      if (rc == AUTODDL_OK) return rc;
      cudaGetLastError();                                    // launch refused: fall back to one CTA per chain
      clear_error();
    }
    return launch_anyk(d_T, Bp, L, K, d_bp, d_opt_cost, d_strategy, st);
  }
  set_error("chain_dp: K = %d not supported (at most 256)", K);
  return AUTODDL_EINVAL;
}

}  // namespace autoddl
