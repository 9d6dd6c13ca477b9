// Fused (a1) + (a2) + first sweep of (a3) on two mesh levels (K = 36): ONE WARP PER CHAIN, no block barrier.
//
// A warp walks its chain layer by layer.  Per layer it evaluates the cost model in FACTOR form:
//   T[l][i][j] = VP[j] + Esym[A(i)][B(j)]
//     VP[j]      = weight-gradient all-reduce of consumer signature j + 2^50 if j is infeasible
//     Esym[a][b] = R[a][b] + R[dual b][dual a]: forward + backward redistribution (Table 2 :102-108)
//                  between the producer's output state vector a and the consumer's input state vector b
//     A(i), B(j) = state-vector index of producer signature i / consumer signature j (16 = invalid for the layer kind:
//                  zero edge), so a tile holds 36 + 17 x 17 numbers of information
// and then, from those 2.6 KB in shared memory,
//   * writes the 36 x 36 tile to HBM with coalesced 16-byte streaming stores (skipped when no table is wanted),
//   * advances the chain DP  f_l[j] = VP[j] + min_i f_{l-1}[i] + Esym[A(i)][B(j)]  (smallest i on ties, R9): 16 input
//     state classes x 2 row halves on the 32 lanes, columns follow their class,
//   * runs the first Coordinate Descent sweep of the chain's starts (R10): the update of layer l-1 needs the row
//     T[l-1][s_{l-2}][.] (stashed in registers one layer earlier) and the column T[l][.][s_l] = Esym_l[A(.)][B(s_l)] + const.
// Nothing is exchanged between warps: no mbarrier, no bar.sync, no TMA hand-off in the layer loop -- the warps of an SM
// (14-16 of them, one CTA per SM) hide each other's latencies.  After the last layer lane 0 back-tracks the chain from
// byte back-pointers in the warp's shared memory (or in a workspace slice for very long chains).
#include "sbp_builder.cuh"

namespace autoddl {

namespace {

constexpr int FK = 36, FD = 2, FNS = 16, FNC = 9, FSTRIDE = FNC + 1, FCELLS = FK * FK;
constexpr int FNU = 10;                                   // classes of a level's (output state, input state) pair, see below
constexpr int FGZ = 143, FG = 144;                        // G[FGZ] = 0: the edge of an invalid signature / of the first layer
constexpr int kMaxFusedStarts = 8;                        // CD starts per chain whose first sweeps ride along

// Esym[a][b] = R[a][b] + R[dual b][dual a] takes only 10 x 10 distinct values on two mesh levels: a level's pair of states
// (a_d, b_d) enters R only through its walk (slice / reduce-scatter / all-to-all / all-gather steps and the split codes
// between them, sbp_builder.cuh) forward and backward, and the 16 pairs fall into FNU = 10 classes of equal (forward walk,
// backward walk).  A tile therefore carries G[u0][u1]: 9 of the 100 entries are zero (no collective on either level),
// 36 are the sum of two entries of the per-level Table-2 values TAB, 42 of four, 12 of six, 1 of eight.  They are computed
// in order of ascending number of summands, so that a round of 32 lanes loads only what its entries need; the consumers
// (tile expansion, DP, CD) reach G through byte index tables built once per CTA.
// Where an entry lives: position 16 (3 hi(u0) + hi(u1)) + 4 col(u0) + col(u1).  col is a 4-colouring of the classes in
// which the classes (a_d, .) of one producer state differ and so do the classes (., b_d) of one consumer state: the 16
// entries a consumer reads along a row of the tile (fixed a, all b) or along a column lie in 16 different 8-byte bank
// slots.  (Performance only: any injective (col, hi) gives the same results.)
__device__ __constant__ uint8_t c_ucol[FNU] = {0, 2, 1, 3, 1, 0, 2, 1, 0, 3};
__device__ __constant__ uint8_t c_uhi[FNU] = {0, 0, 0, 0, 1, 1, 1, 2, 2, 1};
struct CtaShared {
  SigInfo sig[2][FK];
  uint8_t bcls[2][FK];                                    // per consumer kind: B(j) in 0..16 (16 = invalid for the kind)
  uint8_t ucls[16];                                       // class of a level's (a_d, b_d)
  uint8_t ucol[FNU], uhi[FNU];                            // (copies of c_ucol, c_uhi, c_walk: per-thread indices are slow
  uint32_t walk[16];                                      //  in constant memory)
  uint8_t nnz[FNU * FNU];                                 // per (u0, u1): number of summands
  uint32_t ew[2][FNU * FNU];                              // (set-up scratch: its summand words)
  int32_t nl, nh;                                         // entries of 1..4 summands (ranks 0..nl-1), of more (nl..nl+nh-1)
  uint32_t lslot[3][32];                                  // rank 32 k + lane: four 6-bit TAB slots, position in bits 24..31
  uint32_t hslot[2][32];                                  // rank nl + lane: eight slots, position in bits 24..31 of [1]
  alignas(16) uint8_t DPI[2][2][16][16];                  // [producer kind][row half][input class b][part * 4 + q]: DP rows
  uint32_t XI[2][2][6][32];                               // [producer kind][kind][word][lane]: the 24 cells of the lane's class rows
  alignas(4) uint8_t GI[2][2][FK][FK];                    // [producer kind][kind][i][j]: position of Esym[A(i)][B(j)] in G
};

struct alignas(16) Rec64 {                                 // byte image of autoddl_layer
  int64_t X[5];                                           // M, Kd, N, in_rows, in_cols
  int32_t kind, eb, wgb, wsb, maxr, maxc;
};
static_assert(sizeof(Rec64) == sizeof(autoddl_layer), "Rec64 mirrors autoddl_layer");

template <int NB>                                          // NB = 2: the previous layer's factors stay (second CD sweep)
struct alignas(16) WarpShared {
  int64_t Q[5][4];                                        // M, Kd, N, in_rows, in_cols  x  level subset
  int64_t TAB[2 * FD * FSTRIDE];                          // CG[D][NC+1] then CA[D][NC+1]; [..][NC] = 0
  int64_t WAR[FD][FNC];
  int64_t locW[FNC], locO[FNC];
  alignas(16) int64_t VP[NB][FK];                         // layer l in buffer l & (NB - 1)
  int64_t G[NB][FG];                                      // the distinct values of Esym; [FGZ] = 0
  alignas(16) int64_t f[FK];
  Rec64 rec[8];                                           // ring of layer records, fetched four at a time
};

__device__ __forceinline__ void lexmin_xor(int64_t& bv, int& bi) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
    if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
  }
}

// smallest (value, index) over the warp for 0 <= value and index < 64.  Fast path when every value is below 2^57: the
// key value * 64 + index is reduced as two 32-bit halves with redux.sync (the low half only among the lanes that hold
// the smallest high half); otherwise the shuffle butterfly.  Both are exact.
__device__ __forceinline__ void warp_argmin64(int64_t& bv, int& bi) {
  if (__all_sync(0xffffffffu, (uint64_t)bv < (1ull << 57))) {
    const uint64_t key = ((uint64_t)bv << 6) | (uint32_t)bi;
    const uint32_t hi = (uint32_t)(key >> 32), lo = (uint32_t)key;
    const uint32_t mh = __reduce_min_sync(0xffffffffu, hi);
    const uint32_t ml = __reduce_min_sync(0xffffffffu, hi == mh ? lo : 0xffffffffu);
    const uint64_t m = ((uint64_t)mh << 32) | ml;
    bv = (int64_t)(m >> 6);
    bi = (int)(m & 63);
  } else {
    lexmin_xor(bv, bi);
  }
}

// Everything a CTA needs besides the tile data: facts per (layer kind, signature) -- the only part that depends on the mesh
// --, the layout of G and the byte index tables of its consumers.  All threads of the CTA (nthr of them) call it.
__device__ __forceinline__ void fused_cta_setup(CtaShared& cs, const MeshParams& mp, int tid, int nthr) {
  // ---- once per CTA: facts per (layer kind, signature), the layout of G, the index tables ---------------------------
  fill_sig_table<FD>(cs.sig, mp, tid, nthr);
  if (tid >= 32 && tid < 48) cs.walk[tid - 32] = c_walk.w[tid - 32];
  if (tid >= 64 && tid < 64 + FNU) { cs.ucol[tid - 64] = c_ucol[tid - 64]; cs.uhi[tid - 64] = c_uhi[tid - 64]; }
  if (nthr < 96 && tid < 16) {                       // (a CTA of one or two warps)
    cs.walk[tid] = c_walk.w[tid];
    if (tid < FNU) { cs.ucol[tid] = c_ucol[tid]; cs.uhi[tid] = c_uhi[tid]; }
  }
  if (tid < 32) {                                          // class of (a_d, b_d) = rank of its (forward, backward) walk pair
    const int x = tid & 15;
    const uint32_t key = c_walk.w[x] | c_walk.w[dual_of(x & 3) * 4 + dual_of(x >> 2)] << 11;
    int rep = x;                                           // first pair with the same walks
    for (int y = 15; y >= 0; --y)
      if (__shfl_sync(0xffffffffu, key, y) == key) rep = y;
    const uint32_t firsts = __ballot_sync(0xffffffffu, tid < 16 && rep == x);
    if (tid < 16) cs.ucls[x] = (uint8_t)__popc(firsts & ((1u << rep) - 1));
  }
  for (int x = tid; x < 5 * 32; x += nthr) (&cs.lslot[0][0])[x] = FNC | FNC << 6 | FNC << 12 | FNC << 18;   // zero slots (lslot, hslot)
  __syncthreads();
  constexpr uint32_t kNoSlots = FNC | FNC << 6 | FNC << 12 | FNC << 18;
  // the summands of entry e = (u0, u1), 6 bits each in w0 (first four) and w1; returns their number
  auto entry_slots = [&](int e, uint32_t& w0, uint32_t& w1) -> int {
    w0 = w1 = kNoSlots;
    int n = 0, p0 = -1, p1 = -1;                           // a representative state pair per level
    for (int x = 15; x >= 0; --x) {
      if (cs.ucls[x] == e / FNU) p0 = x;
      if (cs.ucls[x] == e % FNU) p1 = x;
    }
    if (p0 < 0 || p1 < 0) return 0;
    const int a = (p0 >> 2) << 2 | (p1 >> 2), b = (p0 & 3) << 2 | (p1 & 3);
    int idx[3 * FD];
    auto take = [&]() {
#pragma unroll
      for (int q = 0; q < 3 * FD; ++q)
        if (idx[q] != FNC) {
          if (n < 4) w0 ^= (uint32_t)(FNC ^ idx[q]) << (6 * n);
          else if (n < 8) w1 ^= (uint32_t)(FNC ^ idx[q]) << (6 * (n - 4));
          else __trap();
          ++n;
        }
    };
    r_slots<FD>(a, b, idx, cs.walk);
    take();
    r_slots<FD>(dual_vec<FD>(b), dual_vec<FD>(a), idx, cs.walk);
    take();
    return n;
  };
  for (int e = tid; e < FNU * FNU; e += nthr) {
    uint32_t w0, w1;
    cs.nnz[e] = (uint8_t)entry_slots(e, w0, w1);
    cs.ew[0][e] = w0;
    cs.ew[1][e] = w1;
  }
  for (int x = tid; x < 2 * FK; x += nthr) {
    const SigInfo& si = cs.sig[x / FK][x % FK];
    cs.bcls[x / FK][x % FK] = (uint8_t)(si.b_idx >= 0 ? si.b_idx : FNS);
  }
  auto upos = [&](int u0, int u1) -> int { return 16 * (3 * cs.uhi[u0] + cs.uhi[u1]) + 4 * cs.ucol[u0] + cs.ucol[u1]; };
  auto gp = [&](int a, int b) -> int {                     // position of Esym[a][b]; a = 16 / b < 0: invalid signature, zero
    if (a >= FNS || b < 0 || b >= FNS) return FGZ;
    return upos(cs.ucls[(a >> 2) << 2 | (b >> 2)], cs.ucls[(a & 3) << 2 | (b & 3)]);
  };
  for (int x = tid; x < 4 * FCELLS; x += nthr) {
    const int kk = x / FCELLS, i = x % FCELLS / FK, j = x % FK;
    cs.GI[kk >> 1][kk & 1][i][j] = (uint8_t)gp(cs.sig[kk >> 1][i].a_idx, cs.sig[kk & 1][j].b_idx);
  }
  for (int x = tid; x < 2 * 2 * 16 * 16; x += nthr) {
    // DP: lane (b, half) scans rows 18 half + 6 part + r; rows whose level-1 digit r is 2, 4 or 5 share their edge (all
    // output P, or all invalid), so a part has four distinct values q = 0..3 for r = 0, 1, 3, 2
    const int kp = x >> 9, half = x >> 8 & 1, bcl = x >> 4 & 15, part = (x & 15) >> 2, q = x & 3;
    const int row = 18 * half + 6 * part + (q < 2 ? q : (q == 2 ? 3 : 2));
    cs.DPI[kp][half][bcl][x & 15] = (uint8_t)(part < 3 ? gp(cs.sig[kp][row].a_idx, bcl) : FGZ);
  }
  __syncthreads();
  for (int e = tid; e < FNU * FNU; e += nthr) {      // computed in order of ascending number of summands, then (u0, u1)
    const int my_n = cs.nnz[e];
    int rank = 0, nl = 0, nh = 0;
    for (int o = 0; o < FNU * FNU; ++o) {
      const int n = cs.nnz[o];
      if (n >= 1 && n <= 4) ++nl;
      if (n > 4) ++nh;
      if (n >= 1 && (n < my_n || (n == my_n && o < e))) ++rank;
    }
    const uint32_t pos = upos(e / FNU, e % FNU);           // (an entry without summands is never written: it stays 0)
    if (e == 0) { cs.nl = nl; cs.nh = nh; }
    if (my_n >= 1 && my_n <= 4) {
      if (rank >= 96 || (rank < 32 && my_n > 2)) __trap();   // (what the rounds below rely on; holds for this walk table)
      cs.lslot[rank >> 5][rank & 31] = cs.ew[0][e] | pos << 24;
    } else if (my_n > 4) {
      if (rank - nl >= 32) __trap();
      cs.hslot[0][rank - nl] = cs.ew[0][e];
      cs.hslot[1][rank - nl] = cs.ew[1][e] | pos << 24;
    }
  }
  for (int x = tid; x < 4 * 6 * 32; x += nthr) {
    // tile expansion: lane (h, pc), class row n = 3 c0 + t -> row (rep(c0), 3 h + t); bytes 2 n, 2 n + 1 = its two columns
    const int kk = x / 192, w = x % 192 / 32, ln = x % 32, pc = ln & 15, h = ln >> 4;
    uint32_t word = 0;
    for (int by = 0; by < 4; ++by) {
      const int n = (4 * w + by) >> 1, col = 2 * pc + ((4 * w + by) & 1), c0 = n / 3, t = n % 3;
      const int r0 = c0 < 2 ? c0 : (c0 == 2 ? 3 : 2);
      word |= (uint32_t)cs.GI[kk >> 1][kk & 1][r0 * 6 + 3 * h + t][col] << (8 * by);
    }
    cs.XI[kk >> 1][kk & 1][w][ln] = word;
  }
  __syncthreads();
}

// The tables above except `sig` are the same for every mesh, launch and CTA: the first launch on a device also runs
// fused_tables_init_kernel, which leaves them in g_fused_tables and then raises g_fused_ready; a CTA that finds the flag up
// copies 12 KB instead of spending ~18 us computing them (kernels that run before the flag is up compute them as before:
// same values either way).
static __device__ __align__(16) unsigned char g_fused_tables[(sizeof(CtaShared) + 15) / 16 * 16];
static __device__ int g_fused_ready = 0;

__global__ void __launch_bounds__(896) fused_tables_init_kernel(MeshParams mp) {
  extern __shared__ __align__(128) unsigned char fti_raw[];
  CtaShared& cs = *reinterpret_cast<CtaShared*>(fti_raw);
  fused_cta_setup(cs, mp, threadIdx.x, blockDim.x);
  __syncthreads();
  const uint4* src = reinterpret_cast<const uint4*>(fti_raw);
  uint4* dst = reinterpret_cast<uint4*>(g_fused_tables);
  for (int x = threadIdx.x; x < (int)(sizeof(g_fused_tables) / 16); x += blockDim.x) dst[x] = src[x];
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    *reinterpret_cast<volatile int*>(&g_fused_ready) = 1;
  }
}

template <int NB>
__global__ void __launch_bounds__(896, 1)
fused_chain36_kernel(const autoddl_layer* __restrict__ layers, int Bp, int L, MeshParams mp,
                     int64_t* __restrict__ T, int64_t* __restrict__ node, uint8_t* __restrict__ mask,
                     int64_t* __restrict__ opt_cost, int32_t* __restrict__ strategy, uint8_t* __restrict__ bp_glob,
                     const int32_t* __restrict__ cd_init, int cd_S, int32_t* __restrict__ cd_s1, int32_t* __restrict__ cd_s2,
                     int per_warp_bytes) {
  extern __shared__ __align__(128) unsigned char fsm_raw[];
  CtaShared& cs = *reinterpret_cast<CtaShared*>(fsm_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, W = blockDim.x >> 5;
  unsigned char* wbase = fsm_raw + ((sizeof(CtaShared) + 127) & ~(size_t)127) + (size_t)warp * per_warp_bytes;
  using WS = WarpShared<NB>;
  WS& ws = *reinterpret_cast<WS*>(wbase);
  // CD only: the row stash of sweep 2 [cd_S][36] int64, then the strategies of the chain's starts after sweep 1 and
  // sweep 2 [2][cd_S][L] bytes; then the back-pointers [L][K] (or a workspace slice: bp_glob)
  int64_t* cd_stash2 = reinterpret_cast<int64_t*>(wbase + sizeof(WS));
  uint8_t* cd_s = wbase + sizeof(WS) + (cd_init ? (size_t)cd_S * FK * 8 : 0);
  uint8_t* cd_t = cd_s + (size_t)cd_S * L;
  const size_t cd_bytes = cd_init ? (((size_t)2 * cd_S * L + 15) & ~(size_t)15) : 0;
  uint8_t* bp = bp_glob ? bp_glob + ((size_t)blockIdx.x * W + warp) * (size_t)L * FK : cd_s + cd_bytes;   // [L][K]
  const bool two = NB == 2 && cd_s2 != nullptr;            // second CD sweep in this kernel as well (NB = 2 whenever CD rides along)

  // ---- once per CTA: the index tables (from the device-wide copy when it is there) and the facts per signature ------------
  {
    __shared__ int s_ready;
    if (tid == 0) {
      s_ready = *reinterpret_cast<volatile int*>(&g_fused_ready);
      __threadfence();                                     // (the tables are read after the flag)
    }
    __syncthreads();
    if (s_ready) {
      const uint4* src = reinterpret_cast<const uint4*>(g_fused_tables);
      uint4* dst = reinterpret_cast<uint4*>(fsm_raw);
      for (int x = tid; x < (int)(sizeof(g_fused_tables) / 16); x += blockDim.x) dst[x] = __ldcg(src + x);
      __syncthreads();
      fill_sig_table<FD>(cs.sig, mp, tid, blockDim.x);     // the mesh-dependent part: this launch's mesh
      __syncthreads();
    } else {
      fused_cta_setup(cs, mp, tid, blockDim.x);
    }
  }
  const int g_nl = cs.nl, g_nh = cs.nh;

  // ---- once per warp: tile-invariant roles of this lane ---------------------------------------------------------
  auto warp_init = [&]() {                                 // zero slots of TAB, zero entry (and first-layer state) of G
    for (int x = lane; x < NB * FG; x += 32) (&ws.G[0][0])[x] = 0;
    if (lane < 2 * FD) ws.TAB[lane * FSTRIDE + FNC] = 0;
  };
  warp_init();
  // step 1: lane (x, m) for lane < 20
  const int q_x = lane >> 2, q_m = lane & 3;
  // (selects between statically indexed parameters: a per-lane index into the parameter space costs a load per use)
  const uint32_t q_sub = (uint32_t)(q_m == 0 ? mp.sub[0] : (q_m == 1 ? mp.sub[1] : (q_m == 2 ? mp.sub[2] : mp.sub[3])));
  const uint64_t q_magic = q_m == 0 ? mp.magic_sub[0] : (q_m == 1 ? mp.magic_sub[1] : (q_m == 2 ? mp.magic_sub[2] : mp.magic_sub[3]));
  // every level size a power of two (the usual machine): ceil(n / d) is an add and a shift
  const bool pow2 = ((mp.size[0] & (mp.size[0] - 1)) | (mp.size[1] & (mp.size[1] - 1))) == 0;
  const int q_sh = 31 - __clz((int)q_sub);
  // step 2: lanes 0..17 = (level, split configuration) for the input tensor and the weight gradient; lanes 18..26 = local sizes
  const int role_i = lane < 18 ? lane : lane - 18;
  const int role_d = lane < 18 ? role_i / FNC : 0, role_cfg = role_i % FNC;
  int role_m0 = 0, role_m1 = 0;
  cfg_masks<FD>(role_cfg, role_m0, role_m1);
  const int64_t r_p = role_d ? mp.size[1] : mp.size[0], r_alpha = role_d ? mp.alpha[1] : mp.alpha[0],
                r_beta = role_d ? mp.beta[1] : mp.beta[0];
  const uint64_t r_magic = role_d ? mp.magic_size[1] : mp.magic_size[0];
  const int r_sh = 31 - __clz((int)r_p);
  auto cdiv_p = [&](int64_t n) -> int64_t { return pow2 ? (n + r_p - 1) >> r_sh : cdiv_magic(n, (uint32_t)r_p, r_magic); };
  const int64_t cap_layer = mp.mem_cap / L;
  const bool capped = mp.mem_cap != 0;                     // no cap: the memory model is not evaluated
  // chain DP: lane (b, half)
  const int dp_b = lane & 15, dp_h = lane >> 4;

  const int nslots = gridDim.x * W;
  for (int p = warp * gridDim.x + blockIdx.x; p < Bp; p += nslots) {
    const autoddl_layer* chain = layers + (size_t)p * L;
    // Layer records: 256-byte groups of four consecutive records per request (16 lanes x 16 bytes; host-mapped inputs are
    // read over PCIe, where small requests are what costs), into a ring of eight, one group (four layers) ahead.
    auto stage4 = [&](int l4) {                              // records l4 .. l4 + 3 -> slots (l4 .. l4 + 3) & 7
      const int l = l4 + (lane >> 2);
      if (lane < 16 && l < L)
        cp_async16(reinterpret_cast<unsigned char*>(&ws.rec[l & 7]) + 16 * (lane & 3),
                   reinterpret_cast<const unsigned char*>(chain + l) + 16 * (lane & 3));
    };
    stage4(0);
    stage4(4);
    int kind_prev = 0, kind_pp = 0;                          // kinds of layers l - 1 and l - 2
    const bool cd = cd_init != nullptr;
    if (cd) {
      for (int x = lane; x < cd_S * L; x += 32) cd_s[x] = (uint8_t)cd_init[(size_t)p * cd_S * L + x];
    }

    for (int l = 0; l < L; ++l) {
      if ((l & 3) == 0) {
        if (lane < 16) cp_async_wait_all();                  // the group of this layer has landed
        __syncwarp();
        if (l >= 4) stage4(l + 4);                           // its slots held layers l-4 .. l-1: done
      }
      const Rec64& rec = ws.rec[l & 7];
      const int kind = rec.kind;
      if (l == 0) kind_prev = kind;                          // no producer: any valid kind (E(0) = 0)
      const size_t tile = (size_t)p * L + l;
      int64_t* const Gc = ws.G[l & (NB - 1)];
      int64_t* const VPc = ws.VP[l & (NB - 1)];
      const int64_t* const Gp = ws.G[(l & (NB - 1)) ^ (NB - 1)];          // layer l - 1 (NB = 2)
      const int64_t* const VPp = ws.VP[(l & (NB - 1)) ^ (NB - 1)];

      // ---- 1. Q[x][m] = ceil(extent x / product of the levels in m) -------------------------------------------------
      if (lane < 20) ws.Q[q_x][q_m] = pow2 ? (rec.X[q_x] + q_sub - 1) >> q_sh : cdiv_magic(rec.X[q_x], q_sub, q_magic);
      __syncwarp();

      // ---- 2. Table 2 per level and split configuration -------------------------------------------
      if (lane < 18) {
        if (l > 0) {                                         // the layer's input tensor: gather / scatter and all-to-all
          const int64_t n = ws.Q[3][role_m0] * ws.Q[4][role_m1] * (int64_t)rec.eb;
          int64_t cg = 0, ca = 0;
          if (r_p > 1) {
            cg = mp.accum * ((r_p - 1) * (r_alpha + cdiv_p(n) * r_beta));
            ca = mp.accum * ((r_p - 1) * r_alpha + n * r_beta);          // R25: once per micro-batch
          }
          ws.TAB[role_d * FSTRIDE + role_cfg] = cg;
          ws.TAB[(FD + role_d) * FSTRIDE + role_cfg] = ca;
        }
        if (kind == AUTODDL_GEMM) {                          // weight gradient: the AllReduce row
          const int64_t n = ws.Q[1][role_m0] * ws.Q[2][role_m1] * (int64_t)rec.wgb;
          ws.WAR[role_d][role_cfg] =
              r_p > 1 ? (2 * r_p - 1) * r_alpha + 2 * (r_p - 1) * cdiv_p(n) * r_beta : 0;
        }
      } else if (lane < 27 && capped) {                      // local sizes of W and O: the memory model only
        ws.locW[role_cfg] = ws.Q[1][role_m0] * ws.Q[2][role_m1];
        ws.locO[role_cfg] = ws.Q[0][role_m0] * ws.Q[2][role_m1];
      }
      __syncwarp();

      // ---- 3. VP[j] (node cost + penalty) and R[a][b] (zero for the first layer: no producer) -------------------------
#pragma unroll
      for (int j0 = 0; j0 < 64; j0 += 32) {
        const int j = j0 + lane;
        if (j < FK) {
          const SigInfo si = cs.sig[kind][j];
          int64_t v = 0, mem = 0;
          if (si.valid) {
            if (kind == AUTODDL_GEMM) {
#pragma unroll
              for (int d = 0; d < FD; ++d)
                if (si.wB >> d & 1) v += ws.WAR[d][si.cfgW];
            }
            if (capped) {                                    // R6: weight state + input + output of the layer
              if (kind == AUTODDL_GEMM) mem = ws.locW[si.cfgW] * (int64_t)rec.wsb;
              mem += (ws.Q[3][si.mI0] * ws.Q[4][si.mI1] + ws.locO[si.cfgO]) * (int64_t)rec.eb;
            }
          }
          const bool ok = si.valid && si.allowed && si.rowsplit <= rec.maxr && si.colsplit <= rec.maxc &&
                          (!capped || mem <= cap_layer);
          VPc[j] = v + (ok ? 0 : AUTODDL_PEN);
          if (node) node[tile * FK + j] = v;
          if (mask) mask[tile * FK + j] = ok ? 1 : 0;
        }
      }
      // G: ranks 0..31 are sums of two TAB entries, 32..nl-1 of at most four, nl..nl+nh-1 (<= 32 of them) of at most eight
      if (l > 0) {
        {
          const uint32_t w = cs.lslot[0][lane];
          Gc[w >> 24] = ws.TAB[w & 63] + ws.TAB[w >> 6 & 63];
        }
#pragma unroll
        for (int k = 1; k < 3; ++k) {
          const uint32_t w = cs.lslot[k][lane];
          const int64_t v = ws.TAB[w & 63] + ws.TAB[w >> 6 & 63] + ws.TAB[w >> 12 & 63] + ws.TAB[w >> 18 & 63];
          if (32 * k + lane < g_nl) Gc[w >> 24] = v;
        }
        if (lane < g_nh) {
          const uint32_t w = cs.hslot[0][lane], x = cs.hslot[1][lane];
          Gc[x >> 24] = ws.TAB[w & 63] + ws.TAB[w >> 6 & 63] + ws.TAB[w >> 12 & 63] + ws.TAB[w >> 18 & 63] +
                        ws.TAB[x & 63] + ws.TAB[x >> 6 & 63] + ws.TAB[x >> 12 & 63] + ws.TAB[x >> 18 & 63];
        }
      } else {
        for (int x = lane; x < FG; x += 32) Gc[x] = 0;        // the first layer has no producer
      }
      __syncwarp();

      // ---- 4. the tile: T[i][j] = VP[j] + Esym[A(i)][B(j)], 16-byte streaming stores --------------------------------------
      // Columns 0..31: lane (h, pc) owns the column pair (2 pc, 2 pc + 1) -- its VP pair and B classes stay in registers --
      // and the rows whose level-1 digit is 3 h + t, t = 0..2.  Rows whose digits agree up to the classes {0},{1},{3},
      // {2,4,5} are identical (signatures 2, 4, 5 all output P, or are all invalid for ATTN), so a value pair is computed
      // once per class row and stored to its 1 or 3 member rows: 12 gathers for 18 stores per lane; a half-warp store
      // covers 256 contiguous bytes.  Columns 32..35: one lane per row, 32 contiguous bytes each.
      if (T) {
        int64_t* out = T + tile * FCELLS;
        {
          const int pc = lane & 15, h = lane >> 4;
          const longlong2 vp = *reinterpret_cast<const longlong2*>(&VPc[2 * pc]);
          const uint32_t* xi = &cs.XI[kind_prev][kind][0][lane];
          uint32_t xw[6];
#pragma unroll
          for (int w = 0; w < 6; ++w) xw[w] = xi[32 * w];
          int64_t* o = out + (3 * h) * FK + 2 * pc;
#pragma unroll
          for (int c0 = 0; c0 < 4; ++c0) {
            const int r0 = c0 < 2 ? c0 : (c0 == 2 ? 3 : 2);  // representative level-0 digit: 0, 1, 3, 2 (= 4 = 5)
#pragma unroll
            for (int t = 0; t < 3; ++t) {
              const int n = 3 * c0 + t;
              const uint32_t pr = xw[n >> 1] >> (16 * (n & 1));
              const longlong2 v = make_longlong2(vp.x + Gc[pr & 255], vp.y + Gc[pr >> 8 & 255]);
              __stcs(reinterpret_cast<longlong2*>(o + (r0 * 6 + t) * FK), v);
              if (c0 == 3) {
                __stcs(reinterpret_cast<longlong2*>(o + (4 * 6 + t) * FK), v);
                __stcs(reinterpret_cast<longlong2*>(o + (5 * 6 + t) * FK), v);
              }
            }
          }
        }
        {
          // columns 32..35: lane (class row (c0, c1), column pair) computes its 16 bytes once and stores them to the 1, 3
          // or 9 rows of the class
          const int c0 = lane >> 3, c1 = lane >> 1 & 3, cp = 32 + 2 * (lane & 1);
          const int d0 = c0 < 2 ? c0 : (c0 == 2 ? 3 : 2), d1 = c1 < 2 ? c1 : (c1 == 2 ? 3 : 2);
          const longlong2 vp = *reinterpret_cast<const longlong2*>(&VPc[cp]);
          const uint32_t gi = *reinterpret_cast<const uint16_t*>(&cs.GI[kind_prev][kind][d0 * 6 + d1][cp]);
          const longlong2 v = make_longlong2(vp.x + Gc[gi & 255], vp.y + Gc[gi >> 8]);
          int64_t* o = out + cp;
#pragma unroll
          for (int m0 = 0; m0 < 3; ++m0) {
#pragma unroll
            for (int m1 = 0; m1 < 3; ++m1) {
              const int r0 = m0 == 0 ? d0 : 3 + m0, r1 = m1 == 0 ? d1 : 3 + m1;          // class 3 = digits 2, 4, 5
              if ((m0 == 0 || c0 == 3) && (m1 == 0 || c1 == 3)) __stcs(reinterpret_cast<longlong2*>(o + (r0 * 6 + r1) * FK), v);
            }
          }
        }
      }

      // ---- 5. chain DP (R9): f_l[j] = VP[j] + min_i f_{l-1}[i] + Esym[A(i)][B(j)], smallest i on ties -----------------
      int64_t* fn = ws.f;
      if (l == 0) {
        for (int j = lane; j < FK; j += 32) fn[j] = VPc[j];            // f_0[j] = T[0][0][j]
      } else {
        const int64_t* f = ws.f;
        const uint4 dq = *reinterpret_cast<const uint4*>(&cs.DPI[kind_prev][dp_h][dp_b][0]);
        const int64_t* fh = f + 18 * dp_h;
        int64_t pb[3];
        int pa[3];
#pragma unroll
        for (int part = 0; part < 3; ++part) {             // three independent chains of six rows, merged in row order
          const uint32_t dw = part == 0 ? dq.x : (part == 1 ? dq.y : dq.z);
          int64_t tv[6], fv[6];
          tv[0] = Gc[dw & 255];
          tv[1] = Gc[dw >> 8 & 255];
          tv[3] = Gc[dw >> 16 & 255];
          tv[2] = tv[4] = tv[5] = Gc[dw >> 24];            // level-1 digits 2, 4, 5: the same edge
#pragma unroll
          for (int r = 0; r < 6; r += 2) {
            const longlong2 f2 = *reinterpret_cast<const longlong2*>(fh + 6 * part + r);
            fv[r] = f2.x;
            fv[r + 1] = f2.y;
          }
          int64_t b = fv[0] + tv[0];
          int ba = 6 * part;
#pragma unroll
          for (int r = 1; r < 6; ++r) {
            const int64_t v = fv[r] + tv[r];
            if (v < b) { b = v; ba = 6 * part + r; }
          }
          pb[part] = b;
          pa[part] = ba;
        }
        int64_t best = pb[0];
        int a = pa[0];
        if (pb[1] < best) { best = pb[1]; a = pa[1]; }
        if (pb[2] < best) { best = pb[2]; a = pa[2]; }
        a += 18 * dp_h;
        {
          const int64_t o = __shfl_down_sync(0xffffffffu, best, 16);
          const int oa = __shfl_down_sync(0xffffffffu, a, 16);
          if (o < best) { best = o; a = oa; }              // rows 18..35 into rows 0..17: strict '<'
        }
        // consumer signatures that are invalid for the layer kind (class 16) have a zero edge: min_i f[i], smallest i
        int64_t h16 = 0;
        int a16 = 0;
        if (kind != AUTODDL_GEMM) {
          h16 = f[lane];
          a16 = lane;
          if (lane < FK - 32) {
            const int64_t v = f[32 + lane];
            if (v < h16) { h16 = v; a16 = 32 + lane; }
          }
          warp_argmin64(h16, a16);
        }
        __syncwarp();                                        // f_{l-1} has been read by every lane: f_l goes in its place
#pragma unroll
        for (int j0 = 0; j0 < 64; j0 += 32) {
          const int j = j0 + lane;
          const int bj = cs.bcls[kind][j < FK ? j : 0];
          int64_t hb = __shfl_sync(0xffffffffu, best, bj & 15);
          int ha = __shfl_sync(0xffffffffu, a, bj & 15);
          if (bj == FNS) { hb = h16; ha = a16; }
          if (j < FK) {
            fn[j] = VPc[j] + hb;
            bp[(size_t)l * FK + j] = (uint8_t)ha;
          }
        }
      }

      // ---- 6. Coordinate Descent (R10): sweep 1 of layer l-1 and, trailing it by one layer, sweep 2 of layer l-2 --------------
      // Sweep 1's update of layer l-1 takes its row T[l-1][s1_{l-2}][.] from the previous tile's factors (still in the other
      // buffer) and its column T[l][.][s_l] from this tile's.  Sweep 2's update of layer m needs the row T[m][s2_{m-1}][.]
      // (stashed at tile m+1, from the previous layer's factors) and the column T[m+1][.][s1_{m+1}], whose s1_{m+1} is final
      // once sweep 1 has passed layer m+1: at tile m+2, with tile m+1's factors still in the other buffer.  Every layer is
      // re-evaluated in sweep 2: the update of a clean layer returns the value it has, so the result is that of the plain
      // algorithm (61 of the 64 layers of a config-4 chain change in sweep 1: sweep 2 would re-evaluate them all anyway).
      // Lane c (and c + 32) owns candidate c: it alone reads and writes stash2[c], so the stash needs no barrier.
      if (NB == 2 && cd) {
        __syncwarp();
        for (int st = 0; st < cd_S; ++st) {
          uint8_t* sv = cd_s + (size_t)st * L;               // after sweep 1 (starts as the initial strategy)
          uint8_t* tv = cd_t + (size_t)st * L;               // after sweep 2
          int64_t* stash2 = cd_stash2 + st * FK;             // T[l-1][s2_{l-2}][.]: row of sweep 2's next update
          int s1 = 0, s2 = 0;                                // s1_{l-1}, s2_{l-2} as updated at this tile (s_{-1} := 0)
          if (l > 0) {                                       // sweep 1, layer l-1
            const uint8_t* grow = cs.GI[kind_pp][kind_prev][l > 1 ? sv[l - 2] : 0];   // (tile 0's G is zero whatever the row)
            const uint8_t* gcol = &cs.GI[kind_prev][kind][0][sv[l]];                  // column s_l of this tile
            int64_t bv = INT64_MAX;
            int bi = FK;
#pragma unroll
            for (int q = 0; q < 2; ++q) {
              const int c = 32 * q + lane;
              if (c < FK) {
                const int64_t g = VPp[c] + Gp[grow[c]] + Gc[gcol[c * FK]];
                if (g < bv) { bv = g; bi = c; }
              }
            }
            warp_argmin64(bv, bi);
            if (lane == 0) sv[l - 1] = (uint8_t)bi;
            s1 = bi;
          }
          if (two && l > 1) {                                // sweep 2, layer l-2: column from tile l-1 given s1_{l-1}
            const uint8_t* gcol = &cs.GI[kind_pp][kind_prev][0][s1];
            int64_t bv = INT64_MAX;
            int bi = FK;
#pragma unroll
            for (int q = 0; q < 2; ++q) {
              const int c = 32 * q + lane;
              if (c < FK) {
                const int64_t g = stash2[c] + Gp[gcol[c * FK]];
                if (g < bv) { bv = g; bi = c; }
              }
            }
            warp_argmin64(bv, bi);
            if (lane == 0) tv[l - 2] = (uint8_t)bi;
            s2 = bi;
          }
          if (two && l > 0) {                                // sweep 2's next row: T[l-1][s2_{l-2}][.]
            const uint8_t* grow2 = cs.GI[kind_pp][kind_prev][s2];
#pragma unroll
            for (int q = 0; q < 2; ++q) {
              const int c = 32 * q + lane;
              if (c < FK) stash2[c] = VPp[c] + Gp[grow2[c]];
            }
          }
          if (l == L - 1) {                                  // the chain ends: the updates that have no later tile
            const uint8_t* grow = cs.GI[kind_prev][kind][s1];
            int64_t bv = INT64_MAX;
            int bi = FK;
#pragma unroll
            for (int q = 0; q < 2; ++q) {                    // sweep 1, last layer: no right neighbour
              const int c = 32 * q + lane;
              if (c < FK) {
                const int64_t g = VPc[c] + Gc[grow[c]];
                if (g < bv) { bv = g; bi = c; }
              }
            }
            warp_argmin64(bv, bi);
            if (lane == 0) sv[l] = (uint8_t)bi;
            if (two) {
              int s2m = 0;                                   // s2_{L-2}
              if (l > 0) {                                   // sweep 2, layer L-2: column from this (last) tile given s1_{L-1}
                const uint8_t* gcol = &cs.GI[kind_prev][kind][0][bi];
                bv = INT64_MAX;
                bi = FK;
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                  const int c = 32 * q + lane;
                  if (c < FK) {
                    const int64_t g = stash2[c] + Gc[gcol[c * FK]];
                    if (g < bv) { bv = g; bi = c; }
                  }
                }
                warp_argmin64(bv, bi);
                if (lane == 0) tv[l - 1] = (uint8_t)bi;
                s2m = bi;
              }
              const uint8_t* grow2 = cs.GI[kind_prev][kind][s2m];   // sweep 2, last layer
              bv = INT64_MAX;
              bi = FK;
#pragma unroll
              for (int q = 0; q < 2; ++q) {
                const int c = 32 * q + lane;
                if (c < FK) {
                  const int64_t g = VPc[c] + Gc[grow2[c]];
                  if (g < bv) { bv = g; bi = c; }
                }
              }
              warp_argmin64(bv, bi);
              if (lane == 0) tv[l] = (uint8_t)bi;
            }
          }
        }
      }
      __syncwarp();
      kind_pp = kind_prev;
      kind_prev = kind;
    }

    // ---- end of the chain: smallest argmin of f_{L-1}, back-track, results --------------------------------------------
    {
      const int64_t* f = ws.f;
      int64_t bv = f[lane];
      int bi = lane;
      if (lane < FK - 32) {
        const int64_t v = f[32 + lane];
        if (v < bv) { bv = v; bi = 32 + lane; }
      }
      warp_argmin64(bv, bi);
      // back-pointers in the workspace: pull the chain's L x 36 bytes into the warp's (now free) tile state first, so
      // that the dependent walk reads shared memory
      const uint8_t* bw = bp;
      __syncwarp();
      if (bp_glob && (size_t)L * FK <= offsetof(WS, rec)) {
        uint8_t* scratch = reinterpret_cast<uint8_t*>(&ws);
        const uint32_t* src = reinterpret_cast<const uint32_t*>(bp);       // L * 36 bytes: a multiple of 4, slices 4-byte aligned
        uint32_t* dst = reinterpret_cast<uint32_t*>(scratch);
        const int n4 = L * FK / 4;
        for (int x0 = 0; x0 < n4; x0 += 32 * 8) {                          // eight independent loads in flight per lane
          uint32_t v[8];
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const int x = x0 + 32 * q + lane;
            v[q] = x < n4 ? __ldcg(src + x) : 0;
          }
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const int x = x0 + 32 * q + lane;
            if (x < n4) dst[x] = v[q];
          }
        }
        __syncwarp();
        bw = scratch;
      }
      if (lane == 0) {
        int32_t* sp = strategy + (size_t)p * L;
        opt_cost[p] = bv;
        int sidx = bi;
        sp[L - 1] = sidx;
        for (int ll = L - 1; ll >= 1; --ll) {
          sidx = bw[(size_t)ll * FK + sidx];
          sp[ll - 1] = sidx;
        }
      }
      __syncwarp();
      if (bw != bp) warp_init();                           // the next chain expects the zero entries of TAB and G
      if (cd) {
        for (int x = lane; x < cd_S * L; x += 32) {
          cd_s1[(size_t)p * cd_S * L + x] = cd_s[x];
          if (two) cd_s2[(size_t)p * cd_S * L + x] = cd_t[x];
        }
      }
      __syncwarp();
    }
  }
}

int fused_sm_count() {
  int dev = 0, sms = 148;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms = 148;
  return sms;
}

constexpr int kMaxWarps = 28;
constexpr size_t kSmemBudget = 226 * 1024;

// per-warp shared memory: tile factors, DP state, (CD) row stashes and strategies of two sweeps, (optionally) back-pointers
size_t warp_bytes(int32_t L, int32_t S, bool bp_smem) {
  const size_t cd = S > 0 ? (((size_t)2 * S * L + 15) & ~(size_t)15) + (size_t)S * FK * 8 : 0;
  return ((S > 0 ? sizeof(WarpShared<2>) : sizeof(WarpShared<1>)) + cd + (bp_smem ? (size_t)L * FK : 0) + 127) & ~(size_t)127;
}
size_t fixed_bytes() { return (sizeof(CtaShared) + 127) & ~(size_t)127; }

}  // namespace

bool fused_build_dp_supported(const MeshParams& mp, int32_t L) { return mp.ndim == 2 && !mp.fold && L >= 1; }

// largest S for which the first two CD sweeps ride in the fused kernel (row stashes and strategies in shared memory)
bool fused_cd_sweep_supported(int32_t L, int32_t S) {
  return S >= 1 && S <= kMaxFusedStarts && fixed_bytes() + 4 * warp_bytes(L, S, false) <= kSmemBudget;
}

// workspace for the back-pointers [L][36] of the chains in flight (one slice per warp) when they do not fit beside the
// warps' shared memory
size_t fused_bp_bytes(int32_t L) {
  static const int sms = fused_sm_count();                 // host-only query, cached
  return ((size_t)sms * kMaxWarps * L * FK + 255) / 256 * 256 + 256;
}

// Fused (a1) + (a2) for K = 36: tables (d_T may be NULL: no table is written) and the chain DP in one kernel, plus the
// first two CD sweeps of S <= 8 starts per chain (d_cd_s1 / d_cd_s2: strategies after sweep 1 / sweep 2; d_cd_s2 NULL:
// one sweep).  d_bp: fused_bp_bytes(L) of workspace.
int launch_build_dp_fused(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int64_t* d_T,
                          int64_t* d_node, uint8_t* d_mask, int64_t* d_opt_cost, int32_t* d_strategy, uint8_t* d_bp,
                          const int32_t* d_cd_init, int32_t S, int32_t* d_cd_s1, int32_t* d_cd_s2, cudaStream_t st) {
  if ((int64_t)Bp * L > 0x7fffffff) { set_error("Bp*L too large"); return AUTODDL_EINVAL; }
  if (!fused_build_dp_supported(mp, L)) { set_error("fused build+DP needs a 2-level mesh"); return AUTODDL_EINVAL; }
  if (d_cd_init && (!fused_cd_sweep_supported(L, S) || d_cd_s1 == nullptr)) { set_error("fused CD sweep: too many starts"); return AUTODDL_EINVAL; }
  const int cdS = d_cd_init ? S : 0;
  const bool two = d_cd_init != nullptr && d_cd_s2 != nullptr;        // two CD sweeps: the previous layer's factors stay
  const int sms = fused_sm_count();
  const size_t fixed = fixed_bytes();
  // one CTA per SM on every SM; warps per CTA: the fewest that reach the minimal number of rounds of chains per warp
  const int grid = Bp < sms ? Bp : sms;
  int wmax = (int)((kSmemBudget - fixed) / warp_bytes(L, cdS, false));
  if (wmax > kMaxWarps) wmax = kMaxWarps;
  if (wmax < 1) { set_error("fused build+DP: chain too long for shared memory"); return AUTODDL_EINVAL; }
  const int rounds = (Bp + grid * wmax - 1) / (grid * wmax);
  int W = (Bp + grid * rounds - 1) / (grid * rounds);
  if (W > wmax) W = wmax;
  if (W < 1) W = 1;
  const bool bp_smem = fixed + (size_t)W * warp_bytes(L, cdS, true) <= kSmemBudget;   // else a workspace slice per warp
  if (!bp_smem && d_bp == nullptr) { set_error("fused build+DP: back-pointer workspace missing"); return AUTODDL_EWORK; }
  const size_t per_warp = warp_bytes(L, cdS, bp_smem);
  const size_t smem = fixed + (size_t)W * per_warp;
  {
    // first launch on this device: also leave the mesh-independent index tables in device memory for every later CTA (the
    // kernels of this stream are ordered behind it; kernels of other streams that start earlier compute the tables themselves)
    static bool launched[64];
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64 && !__atomic_load_n(&launched[dev], __ATOMIC_ACQUIRE)) {
      ADL_CUDA_CHECK(cudaFuncSetAttribute(fused_tables_init_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(CtaShared) + 128));
      fused_tables_init_kernel<<<1, 896, sizeof(CtaShared) + 128, st>>>(mp);
      ADL_CUDA_CHECK(cudaGetLastError());
      __atomic_store_n(&launched[dev], true, __ATOMIC_RELEASE);
    }
  }
  auto kern = cdS > 0 ? fused_chain36_kernel<2> : fused_chain36_kernel<1>;   // CD reads the previous layer's factors
  ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<grid, W * 32, smem, st>>>(d_layers, Bp, L, mp, d_T, d_node, d_mask, d_opt_cost, d_strategy, bp_smem ? nullptr : d_bp,
                                   d_cd_init, cdS, d_cd_s1, two ? d_cd_s2 : nullptr, (int)per_warp);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
