// Coordinate Descent for MANY starts per problem ("hundreds of runs with different initial points") by
// table lookup, on two and three mesh levels (K = 36, 216).
//
// The tables have the factor form  T[l][i][j] = VP_l[j] + Esym_l[A(i)][B(j)]  (A, B = producer-output / consumer-input
// state-vector classes, 17 or 65 of them, the last one = "invalid for the layer kind", zero edge).  The CD
// update of layer l (R10)
//     s_l <- smallest-index argmin_c  T[l][s_{l-1}][c] + T[l+1][c][s_{l+1}]
// therefore depends on its neighbours only through a = A(s_{l-1}) and b = B(s_{l+1}): it is a function BR_l(a, b) with
// 17^2 / 65^2 values per layer, the BEST RESPONSE of layer l.  Three kernels:
//   build_factors_kernel<D>   per tile VP[K] and Esym[ES][ES] (steps 1-3 of the table builders, no K x K expansion)
//   best_response_kernel<D>   BRt[l][b][a] = argmin_c VP_l[c] + Esym_l[a][B(c)] + Esym_{l+1}[A(c)][b], one CTA per layer,
//                             stored transposed (for a known right neighbour the candidates of all a are contiguous) as
//                             16-bit entries (c, A(c)): the class the response presents to layer l + 1 rides along
//   cd_lookup_kernel<D>       one warp per (problem, start): the right neighbour of an update is the OLD s_{l+1}, known
//                             when the sweep starts, so the column BRt[l][B(s_{l+1})][.] of 32 layers at a time is
//                             fetched ahead (one lane per layer, cp.async) and the sweep itself is a chain of ONE
//                             shared-memory look-up per layer, (s_l, A(s_l)) = col_l[A(s_{l-1})]; dirty flags as in
//                             coord_descent.cu.
// Trajectory, sweep count and result are those of the plain algorithm on the K x K tables (same argmin, same
// tie-break), which is what the tests compare with the oracle.  Config 5 (K = 216, L = 480, 1024 starts): the gather
// kernel on the 179 MB tables needs 1,330 us, this path 17 MB of factors + 2 MB of best responses.
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

template <int D>
struct FacSmem {
  using F = Fac<D>;
  alignas(16) int64_t E[F::ES * F::ES];                    // R[a][b]; row NS and column NS stay 0
  int64_t TAB[2 * D * F::STRIDE];                          // CG[D][NC+1] then CA[D][NC+1]; [..][NC] = 0
  int64_t Q[5][8];
  int64_t WAR[D][F::NC];
  int64_t locW[F::NC], locO[F::NC];
  RecBuf rec[2];
  SigInfo sig[2][F::K];
  uint8_t slots[F::NS * F::NS][3 * D];                     // table entries whose sum is R[a][b]
};

template <int D>
__global__ void __launch_bounds__(256) build_factors_kernel(const autoddl_layer* __restrict__ layers, int ntiles, int L, MeshParams mp,
                                                            int64_t* __restrict__ Fout) {
  using F = Fac<D>;
  using SM = FacSmem<D>;
  constexpr int K = F::K, NS = F::NS, NC = F::NC, ES = F::ES, STRIDE = F::STRIDE, NT = 256;
  static_assert(D * NC <= 96 && 192 + NC <= NT && (5 << D) <= NT && K <= NT, "role layout");
  extern __shared__ __align__(16) unsigned char fac_raw[];
  SM& sm = *reinterpret_cast<SM*>(fac_raw);
  const int tid = threadIdx.x;

  fill_sig_table<D>(sm.sig, mp, tid, NT);
  for (int x = tid; x < ES * ES; x += NT) sm.E[x] = 0;
  if (tid < 2 * D) sm.TAB[tid * STRIDE + NC] = 0;
  for (int e = tid; e < NS * NS; e += NT) {
    int idx[3 * D];
    r_slots<D>(e / NS, e % NS, idx);
#pragma unroll
    for (int k = 0; k < 3 * D; ++k) sm.slots[e][k] = (uint8_t)idx[k];
  }
  const int q_x = tid >> D, q_m = tid & ((1 << D) - 1);
  const int role_base = tid < 96 ? 0 : (tid < 192 ? 96 : 192);
  const int role_i = tid - role_base;
  const int role_d = role_i / NC, role_cfg = role_i % NC;
  int role_m0 = 0, role_m1 = 0;
  cfg_masks<D>(role_cfg, role_m0, role_m1);
  const int64_t cap_layer = mp.mem_cap / L;

  int tile = blockIdx.x;
  if (tile >= ntiles) return;
  auto stage = [&](int b, int tl) {
    if (tid < 5) {
      const autoddl_layer* cur = layers + tl;
      RecBuf* dst = &sm.rec[b];
      if (tid < 4) cp_async16(reinterpret_cast<unsigned char*>(dst) + 16 * tid, reinterpret_cast<const unsigned char*>(cur) + 16 * tid);
      else cp_async4(&dst->kind_prev, &(tl % L > 0 ? cur - 1 : cur)->kind);
    }
  };
  stage(0, tile);
  cp_async_wait_all();
  __syncthreads();
  int buf = 0;

  for (; tile < ntiles; tile += gridDim.x, buf ^= 1) {
    const int tile_n = tile + gridDim.x;
    stage(buf ^ 1, tile_n < ntiles ? tile_n : tile);
    const int l = tile % L;
    const RecBuf& rec = sm.rec[buf];
    int64_t* out = Fout + (size_t)tile * F::FB;

    // ---- 1. Q[x][m] -----------------------------------------------------------------------------------------
    if (tid < (5 << D)) sm.Q[q_x][q_m] = cdiv_magic(rec.X[q_x], (uint32_t)mp.sub[q_m], mp.magic_sub[q_m]);
    __syncthreads();
    // ---- 2. Table 2 per level and split configuration ------------------------------------------
    if (role_base == 0 && role_i < D * NC) {
      if (l > 0) {
        const int d = role_d;
        const int64_t n = sm.Q[3][role_m0] * sm.Q[4][role_m1] * (int64_t)rec.eb;
        const int64_t p = mp.size[d];
        int64_t cg = 0, ca = 0;
        if (p > 1) {
          cg = mp.accum * ((p - 1) * (mp.alpha[d] + cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d]));
          ca = mp.accum * ((p - 1) * mp.alpha[d] + n * mp.beta[d]);      // R25: once per micro-batch
        }
        sm.TAB[d * STRIDE + role_cfg] = cg;
        sm.TAB[(D + d) * STRIDE + role_cfg] = ca;
      }
    } else if (role_base == 96 && role_i < D * NC) {
      if (rec.kind == AUTODDL_GEMM) {
        const int d = role_d;
        const int64_t n = sm.Q[1][role_m0] * sm.Q[2][role_m1] * (int64_t)rec.wgb;
        const int64_t p = mp.size[d];
        sm.WAR[d][role_cfg] =
            p > 1 ? (2 * p - 1) * mp.alpha[d] + 2 * (p - 1) * cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d] : 0;
      }
    } else if (role_base == 192 && role_i < NC) {
      sm.locW[role_cfg] = sm.Q[1][role_m0] * sm.Q[2][role_m1];
      sm.locO[role_cfg] = sm.Q[0][role_m0] * sm.Q[2][role_m1];
    }
    __syncthreads();
    // ---- 3. VP[j] straight to the factor block; R[a][b] ---------------------------------------------------------
    if (tid < K) {
      const int j = tid;
      const SigInfo si = sm.sig[rec.kind][j];
      int64_t v = 0, mem = 0;
      if (si.valid) {
        if (rec.kind == AUTODDL_GEMM) {
#pragma unroll
          for (int d = 0; d < D; ++d)
            if (si.wB >> d & 1) v += sm.WAR[d][si.cfgW];
          mem = sm.locW[si.cfgW] * (int64_t)rec.wsb;
        }
        mem += (sm.Q[3][si.mI0] * sm.Q[4][si.mI1] + sm.locO[si.cfgO]) * (int64_t)rec.eb;
      }
      const bool ok = si.valid && si.allowed && si.rowsplit <= rec.maxr && si.colsplit <= rec.maxc && (mp.mem_cap == 0 || mem <= cap_layer);
      out[F::HDR + j] = v + (ok ? 0 : AUTODDL_PEN);
    }
    if (tid == 0) { out[0] = rec.kind; out[1] = rec.kind_prev; }
    for (int e = tid; e < NS * NS; e += NT) {
      int64_t c = 0;
      if (l > 0) {
#pragma unroll
        for (int k = 0; k < 3 * D; ++k) c += sm.TAB[sm.slots[e][k]];
      }
      sm.E[(e / NS) * ES + e % NS] = c;
    }
    __syncthreads();
    // ---- 4. Esym[a][b] = R[a][b] + R[dual b][dual a] (forward + backward leg, R5); row / column NS = 0 --------------
    for (int x = tid; x < ES * ES; x += NT) {
      const int a = x / ES, b = x % ES;
      int64_t v = 0;
      if (a < NS && b < NS) v = sm.E[a * ES + b] + sm.E[dual_vec<D>(b) * ES + dual_vec<D>(a)];
      out[F::HDR + K + x] = v;
    }
    if (tid < 5) cp_async_wait_all();
    __syncthreads();                                       // E is rewritten by the next tile; publishes the next record
  }
}

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

template <int D>
struct BrSmem {
  using F = Fac<D>;
  alignas(16) int64_t VP[F::K];
  alignas(16) int64_t El[F::ES * F::ES + 1];               // Esym of layer l (overwritten by the class minima W, as keys)
  alignas(16) int64_t Er[F::ES * F::ES + 1];               // Esym of layer l + 1
  SigInfo sig[2][F::K];
  uint8_t acls[2][F::K], bcls[2][F::K];
  uint8_t mstart[2][F::ES + 1], mlist[2][F::K];            // per kind: the candidates of every producer class alpha, ascending
};

// BRt[l][b][a] = smallest-index argmin_c  VP_l[c] + Esym_l[a][B(c)] + Esym_{l+1}[A(c)][b].
// The right term depends on c only through alpha = A(c), so the minimum splits:
//   W[a][alpha] = min_{c : A(c) = alpha} VP_l[c] + Esym_l[a][B(c)]   (smallest c on ties),
//   BR(a, b)    = the c of argmin_alpha  W[a][alpha] + Esym_{l+1}[alpha][b]   (ties: the smaller c).
// 65 x 216 + 65 x 65 x 65 operations per layer instead of 65 x 65 x 216 at K = 216.
template <int D>
__global__ void __launch_bounds__(512) best_response_kernel(const int64_t* __restrict__ Fin, int ntiles, int L, MeshParams mp,
                                                            uint8_t* __restrict__ BRt) {
  using F = Fac<D>;
  constexpr int K = F::K, ES = F::ES, CS = F::CS, NT = 512, NW = (ES * ES + NT - 1) / NT;
  constexpr int64_t kNone = (int64_t)1 << 61;             // no candidate in the class (real sums stay below 2^53)
  constexpr int64_t kNoneKey = (int64_t)1 << 62;
  extern __shared__ __align__(16) unsigned char br_raw[];
  BrSmem<D>& sm = *reinterpret_cast<BrSmem<D>*>(br_raw);
  const int tid = threadIdx.x;
  fill_sig_table<D>(sm.sig, mp, tid, NT);
  __syncthreads();
  fill_classes<D>(sm.acls, sm.bcls, sm.sig, tid, NT);
  __syncthreads();
  // candidates per producer class, ascending: count, prefix, fill -- a warp per (kind, class), 32 candidates per ballot
  const int lane = tid & 31, warp = tid >> 5;
  for (int pr = warp; pr < 2 * ES; pr += NT / 32) {
    const int kind = pr / ES, al = pr % ES;
    int n = 0;
    for (int c0 = 0; c0 < K; c0 += 32) n += __popc(__ballot_sync(0xffffffffu, c0 + lane < K && sm.acls[kind][c0 + lane] == al));
    if (lane == 0) sm.mstart[kind][al + 1] = (uint8_t)n;   // (counts for now)
  }
  __syncthreads();
  if (tid < 2) {
    int n = 0;
    sm.mstart[tid][0] = 0;
    for (int al = 0; al < ES; ++al) { n += sm.mstart[tid][al + 1]; sm.mstart[tid][al + 1] = (uint8_t)n; }
  }
  __syncthreads();
  for (int pr = warp; pr < 2 * ES; pr += NT / 32) {
    const int kind = pr / ES, al = pr % ES;
    int n = sm.mstart[kind][al];
    for (int c0 = 0; c0 < K; c0 += 32) {
      const bool mine = c0 + lane < K && sm.acls[kind][c0 + lane] == al;
      const uint32_t m = __ballot_sync(0xffffffffu, mine);
      if (mine) sm.mlist[kind][n + __popc(m & ((1u << lane) - 1))] = (uint8_t)(c0 + lane);
      n += __popc(m);
    }
  }
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int l = tile % L;
    const bool has_right = l < L - 1;
    const int64_t* f = Fin + (size_t)tile * F::FB;
    __syncthreads();
    // the factor blocks of layers l and l + 1, 16 bytes per request, asynchronously (HDR + K is even: 16-byte aligned)
    static_assert((F::HDR + K) % 2 == 0 && F::FB % 2 == 0 && K % 2 == 0, "16-byte pieces");
    for (int x = tid; x < K / 2; x += NT) cp_async16(&sm.VP[2 * x], f + F::HDR + 2 * x);
    for (int x = tid; x < (ES * ES + 1) / 2; x += NT) {
      cp_async16(&sm.El[2 * x], f + F::HDR + K + 2 * x);
      if (has_right) cp_async16(&sm.Er[2 * x], f + F::FB + F::HDR + K + 2 * x);
      else { sm.Er[2 * x] = 0; sm.Er[2 * x + 1] = 0; }
    }
    cp_async_wait_all();
    __syncthreads();
    const int kind = (int)f[0];                            // kind of layer l: classes B(c) of the candidates as consumers of
    const uint8_t* bc = sm.bcls[kind];                     // tile l and A(c) as producers of tile l + 1
    const uint8_t* ms = sm.mstart[kind];
    const uint8_t* ml = sm.mlist[kind];
    // W[a][alpha] = min over the candidates c of producer class alpha of VP[c] + El[a][B(c)], smallest c on ties, as the key
    // W * 256 + c (sums stay below 2^53) -- into registers (the rows of El are still being read), then over El.  A warp
    // takes one class alpha and 32 rows a: its lanes walk the same candidate list.  The candidates that are invalid for
    // the kind (class ES - 1) all carry 2^50 and the zero edge: the first one wins.
    int64_t wk[NW];
#pragma unroll
    for (int q = 0; q < NW; ++q) {
      const int x = tid + q * NT;
      wk[q] = kNoneKey;
      if (x < ES * ES) {
        const int al = x / ES, a = x % ES;
        const int64_t* row = sm.El + a * ES;
        const int m0 = ms[al], m1 = al == ES - 1 ? (ms[al + 1] > m0 ? m0 + 1 : m0) : ms[al + 1];
        int64_t wv = kNone;
        int wc = 255;
        for (int m = m0; m < m1; ++m) {
          const int c = ml[m];
          const int64_t g = sm.VP[c] + row[bc[c]];
          if (g < wv) { wv = g; wc = c; }
        }
        if (wc != 255) wk[q] = wv << 8 | wc;
      }
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NW; ++q) {
      const int x = tid + q * NT;
      if (x < ES * ES) {
        sm.El[x % ES * ES + x / ES] = wk[q];
        sm.Er[x] <<= 8;                                    // the right edge in key units
      }
    }
    __syncthreads();
    // BR[a][b] = argmin over alpha of W[a][alpha] + Er[alpha][b]: (value, candidate) lexicographic = plain min of the keys
    // (an empty class carries 2^62: it never wins).  Thread (ta, tb) owns the R x R outputs (ta + T i, tb + T j): R loads
    // of W and R of Er per alpha for R^2 sums; lanes run along b: the Er loads are conflict-free, the W loads broadcasts.
    const uint8_t* ac = sm.acls[kind];
    uint8_t* out = BRt + (size_t)tile * ES * CS;
    constexpr int R = D == 3 ? 3 : 1, T = (ES + R - 1) / R;
    static_assert(T * T <= NT, "one pass");
    if (tid < T * T) {
      const int ta = tid / T, tb = tid % T;
      int64_t best[R][R];
      int ao[R], bo[R];
#pragma unroll
      for (int i = 0; i < R; ++i) {
        ao[i] = (ta + T * i < ES ? ta + T * i : ES - 1) * ES;        // (clamped: the value is dropped below)
        bo[i] = tb + T * i < ES ? tb + T * i : ES - 1;
#pragma unroll
        for (int j = 0; j < R; ++j) best[i][j] = INT64_MAX;
      }
#pragma unroll 5
      for (int al = 0; al < ES; ++al) {
        int64_t wv[R], cv[R];
#pragma unroll
        for (int i = 0; i < R; ++i) { wv[i] = sm.El[ao[i] + al]; cv[i] = sm.Er[al * ES + bo[i]]; }
#pragma unroll
        for (int i = 0; i < R; ++i)
#pragma unroll
          for (int j = 0; j < R; ++j) {
            const int64_t g = wv[i] + cv[j];
            best[i][j] = g < best[i][j] ? g : best[i][j];
          }
      }
      // the entry: the candidate and the producer class it presents to layer l + 1 (the next look-up's row)
#pragma unroll
      for (int i = 0; i < R; ++i)
#pragma unroll
        for (int j = 0; j < R; ++j) {
          const int a = ta + T * i, b2 = tb + T * j;
          if (a < ES && b2 < ES) {
            const int arg = (int)(best[i][j] & 255);
            reinterpret_cast<uint16_t*>(out + b2 * CS)[a] = (uint16_t)(arg | ac[arg] << 8);
          }
        }
    }
  }
}

template <int D>
__global__ void __launch_bounds__(128) cd_lookup_kernel(const int64_t* __restrict__ Fin, const uint8_t* __restrict__ BRt, int Bp, int L,
                                                        int S, MeshParams mp, const int32_t* __restrict__ init, int max_sweeps,
                                                        int64_t* __restrict__ cost, int32_t* __restrict__ strategy,
                                                        int32_t* __restrict__ sweeps, int per_warp_bytes) {
  using F = Fac<D>;
  constexpr int K = F::K, ES = F::ES, CS = F::CS;
  extern __shared__ __align__(16) unsigned char cdl_raw[];
  struct Shared { SigInfo sig[2][K]; uint8_t acls[2][K], bcls[2][K]; };
  Shared& cs = *reinterpret_cast<Shared*>(cdl_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, W = blockDim.x >> 5;
  fill_sig_table<D>(cs.sig, mp, tid, blockDim.x);
  __syncthreads();
  fill_classes<D>(cs.acls, cs.bcls, cs.sig, tid, blockDim.x);
  __syncthreads();
  const size_t ps = (size_t)blockIdx.x * W + warp;
  if (ps >= (size_t)Bp * S) return;
  const size_t p = ps / S;
  unsigned char* wb = cdl_raw + ((sizeof(Shared) + 15) & ~(size_t)15) + (size_t)warp * per_warp_bytes;
  uint8_t* chunk = wb;                                     // [2][32][CS] best-response columns of 32 layers, double buffered
  uint8_t* s = chunk + 2 * 32 * CS;                        // [L] strategy
  uint8_t* kinds = s + L;                                  // [L] layer kinds
  uint8_t* dirty = kinds + L;                              // [L]
  const int64_t* Fp = Fin + p * (size_t)L * F::FB;
  const uint8_t* Bp_ = BRt + p * (size_t)L * ES * CS;
  for (int l = lane; l < L; l += 32) {
    s[l] = (uint8_t)init[ps * L + l];
    kinds[l] = (uint8_t)Fp[(size_t)l * F::FB];
    dirty[l] = 1;
  }
  __syncwarp();

  // column of layer l for the CURRENT right neighbour (old s_{l+1}: it is not touched before layer l + 1's own turn)
  auto fetch = [&](int l0, int b) {                        // lane i -> layer l0 + i -> chunk[b][i][0 .. CS), asynchronously
    const int l = l0 + lane;
    if (l < L) {
      const int bcl = l < L - 1 ? cs.bcls[kinds[l + 1]][s[l + 1]] : 0;
      const unsigned char* src = Bp_ + ((size_t)l * ES + bcl) * CS;
      unsigned char* dst = chunk + ((size_t)b * 32 + lane) * CS;
#pragma unroll
      for (int q = 0; q < CS / 16; ++q) cp_async16(dst + 16 * q, src + 16 * q);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  int nsweeps = 0;
  for (;;) {
    bool changed = false;
    bool carry = false;                                    // the previous layer changed in this sweep: this one is dirty now
    int aprev = 0;                                         // A(s_{l-1}): the row of the next look-up (every lane tracks it)
    int cb = 0;
    bool have = false;                                     // chunk cb holds the columns of the current block of 32 layers
    for (int l0 = 0; l0 < L; l0 += 32) {
      const int n = L - l0 < 32 ? L - l0 : 32;
      // the block's state in registers (lane i <-> layer l0 + i): its signature and the producer class it presents to
      // the next layer; every lane walks the block on uniform values, shared memory is only read during the walk
      int sreg = lane < n ? s[l0 + lane] : 0;
      int areg = lane < n ? cs.acls[kinds[l0 + lane]][sreg] : 0;
      const unsigned dmask = __ballot_sync(0xffffffffu, lane < n && dirty[l0 + lane]);
      if (dmask == 0 && !carry) {                          // nothing to do in this block: nothing can become dirty either
        aprev = __shfl_sync(0xffffffffu, areg, n - 1);
        if (have) asm volatile("cp.async.wait_group 0;" ::: "memory");   // a fetch made for this block lands before its buffer is reused
        have = false;
        continue;
      }
      if (!have) fetch(l0, cb);
      const bool ahead = l0 + 32 < L;
      if (ahead) fetch(l0 + 32, cb ^ 1);                   // the next block's columns travel while this one is walked
      if (ahead) asm volatile("cp.async.wait_group 1;" ::: "memory"); else asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncwarp();
      const uint16_t* colb = reinterpret_cast<const uint16_t*>(chunk + (size_t)cb * 32 * CS);
      // Walk from the first layer that has to be re-evaluated to the end of the block, evaluating EVERY layer on the way:
      // a clean layer's update is a function of unchanged neighbours and returns the value it already has, so nothing
      // depends on whether the previous layer changed and the chain is ONE shared-memory read per layer -- the entry holds
      // the best response and the class it presents to the next layer.  Lane i keeps the entry of its own layer.
      const int i0 = carry ? 0 : __ffs(dmask) - 1;
      if (i0 > 0) aprev = __shfl_sync(0xffffffffu, areg, i0 - 1);
      int mine = sreg | areg << 8;
      for (int i = i0; i < n; ++i) {
        const int e = colb[i * (CS / 2) + aprev];          // (layer 0: aprev = 0, and its entries do not depend on the row)
        if (lane == i) mine = e;
        aprev = e >> 8;
      }
      const unsigned chm = __ballot_sync(0xffffffffu, lane < n && (mine & 255) != sreg);
      if (chm) changed = true;
      carry = chm >> (n - 1) & 1;
      const unsigned dnext = chm >> 1;                     // a layer whose right neighbour changed: dirty in the next sweep
      if ((chm & 1) && l0 > 0 && lane == 0) dirty[l0 - 1] = 1;   // (last layer of the previous block, already walked)
      sreg = mine & 255;
      if (lane < n) {
        s[l0 + lane] = (uint8_t)sreg;
        dirty[l0 + lane] = dnext >> lane & 1;
      }
      __syncwarp();
      cb ^= 1;
      have = l0 + 32 < L;
    }
    ++nsweeps;
    if (!changed || nsweeps >= max_sweeps) break;
    __syncwarp();
  }
  __syncwarp();

  // Cost(s) = sum_l T[l][s_{l-1}][s_l] = sum_l VP_l[s_l] + Esym_l[A(s_{l-1})][B(s_l)]   (Esym_0 = 0; s_{-1} := 0)
  int64_t acc = 0;
  for (int l = lane; l < L; l += 32) {
    const int64_t* f = Fp + (size_t)l * F::FB;
    const int sl = s[l];
    const int a = l > 0 ? cs.acls[kinds[l - 1]][s[l - 1]] : 0;
    const int b = cs.bcls[kinds[l]][sl];
    acc += __ldg(f + F::HDR + sl) + __ldg(f + F::HDR + K + a * ES + b);
    strategy[ps * L + l] = sl;
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
  if (lane == 0) {
    cost[ps] = acc;
    sweeps[ps] = nsweeps;
  }
}

// ---- chain DP (R9) of FEW LONG chains, parallel over the layers ---------------------------------------------------------
// One chain is a sequential recurrence, and a CTA (or an 8-CTA cluster on the tables, chain_dp_cluster.cu) needs about a
// microsecond per layer whatever it does: 441 us for the 480 layers of config 5.  In class space the recurrence is
//   g_l[a'] = min_a g_{l-1}[a] + M_l[a][a'],   g_l[a] = min_{j : A(j) = a} f_l[j],
//   M_l[a][a'] = min_{j : A(j) = a'} VP_l[j] + Esym_l[a][B(j)]                      (17 x 17 / 65 x 65 numbers per layer),
// a chain of min-plus vector-matrix products, which is associative and exact on integers.  So:
//   1. class_matrix_kernel   M_l for every layer (a CTA per layer; M_0's rows all equal g_0 because Esym_0 = 0)
//   2. chunk_product_kernel  Q_c = M_{t_c + 1} (x) ... (x) M_{t_c + len}, t_c = c len  (a CTA per chunk, len - 1 products)
//   3. chunk_prefix_kernel   V_0 = g_0, V_{c+1} = V_c (x) Q_c = g_{t_{c+1}}             (a CTA per chain, C - 1 short steps)
//   4. chunk_dp_kernel       a CTA per chunk restarts the ordinary DP from g_{t_c}: layer t_c + 1 rebuilds f (hence the
//                            smallest index per class), layers t_c + 2 .. t_{c+1} + 1 write their back-pointers exactly as the
//                            sequential DP does (smallest i on ties); the last chunk leaves f_{L-1}'s smallest argmin
//   5. chain_walk_kernel     back-pointers to shared memory, the walk.
// "No signature in the class" is 2^61 (real costs stay below 2^60); products are clamped to it.
constexpr int64_t kInfCls = (int64_t)1 << 61;

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

template <int D>
struct CmSmem {
  using F = Fac<D>;
  alignas(16) int64_t VP[F::K];
  alignas(16) int64_t E[F::ES * F::ES + 1];
  SigInfo sig[2][F::K];
  uint8_t acls[2][F::K], bcls[2][F::K];
  uint8_t mstart[2][F::ES + 1], mlist[2][F::K];
};

// 1. M[tile][a][a'] (row-major, ES x ES int64; matrices are N2P = ES^2 + 1 words apart: 16-byte multiples for the bulk copies)
template <int D>
__global__ void __launch_bounds__(512) class_matrix_kernel(const int64_t* __restrict__ Fin, int ntiles, MeshParams mp,
                                                           int64_t* __restrict__ Mout) {
  using F = Fac<D>;
  constexpr int K = F::K, ES = F::ES, NT = 512, NW = (ES * ES + NT - 1) / NT;
  extern __shared__ __align__(16) unsigned char cm_raw[];
  CmSmem<D>& sm = *reinterpret_cast<CmSmem<D>*>(cm_raw);
  const int tid = threadIdx.x;
  fill_sig_table<D>(sm.sig, mp, tid, NT);
  __syncthreads();
  fill_classes<D>(sm.acls, sm.bcls, sm.sig, tid, NT);
  __syncthreads();
  fill_members<D>(sm.mstart, sm.mlist, sm.acls, tid, NT);
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int64_t* f = Fin + (size_t)tile * F::FB;
    __syncthreads();
    for (int x = tid; x < K / 2; x += NT) cp_async16(&sm.VP[2 * x], f + F::HDR + 2 * x);
    for (int x = tid; x < (ES * ES + 1) / 2; x += NT) cp_async16(&sm.E[2 * x], f + F::HDR + K + 2 * x);
    cp_async_wait_all();
    __syncthreads();
    const int kind = (int)f[0];
    const uint8_t* bc = sm.bcls[kind];
    const uint8_t* ms = sm.mstart[kind];
    const uint8_t* ml = sm.mlist[kind];
    int64_t wv[NW];
#pragma unroll
    for (int q = 0; q < NW; ++q) {                         // a warp takes one class a' and 32 rows a: one member list
      const int x = tid + q * NT;
      wv[q] = kInfCls;
      if (x < ES * ES) {
        const int al = x / ES, a = x % ES;
        const int64_t* row = sm.E + a * ES;
        // (the signatures that are invalid for the kind all carry 2^50 and the zero edge: one of them is enough)
        const int m0 = ms[al], m1 = al == ES - 1 ? (ms[al + 1] > m0 ? m0 + 1 : m0) : ms[al + 1];
        for (int m = m0; m < m1; ++m) {
          const int c = ml[m];
          const int64_t g = sm.VP[c] + row[bc[c]];
          wv[q] = g < wv[q] ? g : wv[q];
        }
      }
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NW; ++q) {
      const int x = tid + q * NT;
      if (x < ES * ES) sm.E[x % ES * ES + x / ES] = wv[q];
    }
    __syncthreads();
    int64_t* out = Mout + (size_t)tile * F::N2P;
    for (int x = tid; x < ES * ES; x += NT) out[x] = sm.E[x];
  }
}

// 2. Q[p][c] = M_{t_c + 1} (x) ... (x) M_{t_c + len} for c = 0 .. C - 2, evaluated from the right: a CTA owns a group of W
// columns of the result, X = M_{t_c + len}[., cols], X <- M_k (x) X for k = t_c + len - 1 .. t_c + 1 -- the column groups of a
// chunk never talk to each other (grid.x = C - 1, grid.y = Bp, grid.z = groups).  One TMA bulk copy per matrix, two in flight.
template <int D>
struct ProdCfg {
  static constexpr int ES = Fac<D>::ES;
  static constexpr int NG = D == 3 ? 5 : 1;                // column groups
  static constexpr int W = (ES + NG - 1) / NG;             // 13 / 17 columns each
  static constexpr int RA = D == 3 ? 3 : 1, RJ = 1;        // outputs per thread: rows a + TA i, columns j + TJ k.  The loop
  static constexpr int TA = (ES + RA - 1) / RA;            // is bound by shared-memory loads (RA + RJ per RA RJ sums) and by the
  static constexpr int TJ = (W + RJ - 1) / RJ;             // 64-bit min (6 instructions); 3 x 1 measured best (3 x 3: too few
  static constexpr int NT = (TA * TJ + 31) / 32 * 32;      // warps on the SM, 1 x 1: twice the loads): 288 / 320 threads
};

template <int D>
__global__ void __launch_bounds__(ProdCfg<D>::NT) chunk_product_kernel(const int64_t* __restrict__ M, int L, int len, int64_t* __restrict__ Q) {
  using F = Fac<D>;
  using PC = ProdCfg<D>;
  constexpr int ES = F::ES, N2P = F::N2P, W = PC::W, RA = PC::RA, RJ = PC::RJ, TA = PC::TA, TJ = PC::TJ, NT = PC::NT;
  extern __shared__ __align__(128) unsigned char cp_raw[];
  int64_t* Ab = reinterpret_cast<int64_t*>(cp_raw);        // two matrix buffers [N2P], then X [2][ES][W]
  int64_t* X = Ab + 2 * N2P;
  __shared__ uint64_t bar[2];
  const int tid = threadIdx.x, c = blockIdx.x, p = blockIdx.y, col0 = blockIdx.z * W;
  const int ncol = col0 + W <= ES ? W : ES - col0;
  const int64_t* Mp = M + ((size_t)p * L + (size_t)c * len) * N2P;         // M_{t_c}; M_{t_c + k} = Mp + k N2P
  if (tid == 0) {
    mbar_init(&bar[0], 1); mbar_init(&bar[1], 1);
    mbar_fence_init();
  }
  __syncthreads();
  const uint64_t pol = policy_evict_first();
  // use u = 0, 1, ..: matrix k = len - u into buffer u & 1
  auto fetch = [&](int u) {                                // thread 0
    if (u < len) {
      mbar_arrive_expect_tx(&bar[u & 1], N2P * 8);
      bulk_g2s(Ab + (u & 1) * N2P, Mp + (size_t)(len - u) * N2P, N2P * 8, &bar[u & 1], pol);
    }
  };
  if (tid == 0) { fetch(0); fetch(1); }
  mbar_wait(&bar[0], 0);
  for (int x = tid; x < ES * W; x += NT) {                 // X = the CTA's columns of M_{t_c + len}
    const int m = x / W, j = x % W;
    X[x] = j < ncol ? Ab[m * ES + col0 + j] : kInfCls;
  }
  __syncthreads();
  if (tid == 0) fetch(2);
  const int ta = tid / TJ, tj = tid % TJ;
  int cur = 0;
  for (int u = 1; u < len; ++u) {
    mbar_wait(&bar[u & 1], (u >> 1) & 1);
    const int64_t* A = Ab + (u & 1) * N2P;
    const int64_t* Xc = X + cur * ES * W;
    int64_t* Xn = X + (cur ^ 1) * ES * W;
    if (ta < TA) {
      int ao[RA], jo[RJ];
      int64_t best[RA][RJ];
#pragma unroll
      for (int i = 0; i < RA; ++i) {
        ao[i] = (ta + TA * i < ES ? ta + TA * i : ES - 1) * ES;        // (clamped: dropped below)
#pragma unroll
        for (int k = 0; k < RJ; ++k) best[i][k] = INT64_MAX;
      }
#pragma unroll
      for (int k = 0; k < RJ; ++k) jo[k] = tj + TJ * k < W ? tj + TJ * k : W - 1;
#pragma unroll 5
      for (int m = 0; m < ES; ++m) {
        int64_t av[RA], xv[RJ];
#pragma unroll
        for (int i = 0; i < RA; ++i) av[i] = A[ao[i] + m];
#pragma unroll
        for (int k = 0; k < RJ; ++k) xv[k] = Xc[m * W + jo[k]];
#pragma unroll
        for (int i = 0; i < RA; ++i)
#pragma unroll
          for (int k = 0; k < RJ; ++k) {
            const int64_t g = av[i] + xv[k];
            best[i][k] = g < best[i][k] ? g : best[i][k];
          }
      }
#pragma unroll
      for (int i = 0; i < RA; ++i)
#pragma unroll
        for (int k = 0; k < RJ; ++k)
          if (ta + TA * i < ES && tj + TJ * k < W) Xn[(ta + TA * i) * W + tj + TJ * k] = best[i][k] < kInfCls ? best[i][k] : kInfCls;
    }
    cur ^= 1;
    __syncthreads();                                       // the matrix buffer has been read, the new X is complete
    if (tid == 0) fetch(u + 2);
  }
  int64_t* out = Q + ((size_t)p * gridDim.x + c) * (ES * F::SQ) + col0;    // rows SQ words apart
  const int64_t* Xc = X + cur * ES * W;
  for (int x = tid; x < ES * W; x += NT)
    if (x % W < ncol) out[x / W * F::SQ + x % W] = Xc[x];
}

// 3. V[p][0] = g_0 (any row of M_0), V[p][c + 1] = V[p][c] (x) Q[p][c]   (one CTA per chain; nq = C - 1 matrices, TMA ring).
// The steps are sequential and short: thread (b, part) of 4 parts per output b takes every fourth a; with rows SQ = 8 mod 16
// words apart the 32 lanes of a load (8 outputs x 4 parts) hit 32 different 8-byte bank slots.
template <int D>
__global__ void __launch_bounds__((Fac<D>::ES * 4 + 31) / 32 * 32) chunk_prefix_kernel(const int64_t* __restrict__ M, int L,
                                                                                    const int64_t* __restrict__ Q, int nq,
                                                                                    int64_t* __restrict__ V) {
  using F = Fac<D>;
  constexpr int ES = F::ES, SQ = F::SQ, QW = ES * SQ, PARTS = 4, ST = 4, NA = (ES + PARTS - 1) / PARTS;
  extern __shared__ __align__(128) unsigned char pf_raw[];
  int64_t* ring = reinterpret_cast<int64_t*>(pf_raw);      // ST matrices
  __shared__ int64_t v[2][ES];
  __shared__ uint64_t full[ST];
  const int tid = threadIdx.x, p = blockIdx.x;
  const int b = tid / PARTS, part = tid % PARTS;
  const int64_t* Qp = Q + (size_t)p * nq * QW;
  if (tid == 0) {
    for (int s2 = 0; s2 < ST; ++s2) mbar_init(&full[s2], 1);
    mbar_fence_init();
  }
  __syncthreads();
  const uint64_t pol = policy_evict_first();
  auto fetch = [&](int c) {                                // thread 0
    if (c < nq) {
      mbar_arrive_expect_tx(&full[c % ST], QW * 8);
      bulk_g2s(ring + (size_t)(c % ST) * QW, Qp + (size_t)c * QW, QW * 8, &full[c % ST], pol);
    }
  };
  if (tid == 0)
    for (int s2 = 0; s2 < ST; ++s2) fetch(s2);
  if (tid < ES) {
    const int64_t g0 = M[(size_t)p * L * F::N2P + tid];
    v[0][tid] = g0;
    V[(size_t)p * (nq + 1) * ES + tid] = g0;
  }
  __syncthreads();
  for (int c = 0; c < nq; ++c) {
    mbar_wait(&full[c % ST], (c / ST) & 1);
    const int64_t* Qc = ring + (size_t)(c % ST) * QW + (b < ES ? b : 0);
    const int64_t* vin = v[c & 1];
    int64_t t[NA];
#pragma unroll
    for (int q = 0; q < NA; ++q) {
      const int a = part + q * PARTS;
      t[q] = a < ES ? vin[a] + Qc[a * SQ] : kInfCls;
    }
    int64_t best = kInfCls;
#pragma unroll
    for (int q = 0; q < NA; ++q) best = t[q] < best ? t[q] : best;
#pragma unroll
    for (int off = 1; off < PARTS; off <<= 1) {
      const int64_t o = __shfl_xor_sync(0xffffffffu, best, off);
      best = o < best ? o : best;
    }
    if (b < ES && part == 0) {
      v[(c & 1) ^ 1][b] = best;
      V[((size_t)p * (nq + 1) + c + 1) * ES + b] = best;
    }
    __syncthreads();
    if (tid == 0) fetch(c + ST);
  }
}

template <int D>
struct CdpSmem {
  using F = Fac<D>;
  static constexpr int ST = D == 3 ? 4 : 8;
  alignas(128) int64_t blk[ST][F::FB];                     // ring of factor blocks (TMA bulk copies)
  uint64_t full[ST];
  int64_t g[F::ES], h[F::ES];
  int32_t gi[F::ES], hi[F::ES];
  SigInfo sig[2][F::K];
  uint8_t acls[2][F::K], bcls[2][F::K];
  uint8_t mstart[2][F::ES + 1], mlist[2][F::K];
};

// 4. the DP of chunk c of chain p, restarted from V[p][c] = g_{t_c} (grid.x = C, grid.y = Bp)
template <int D>
__global__ void __launch_bounds__(Fac<D>::ES * 8 / 32 * 32 + 32) chunk_dp_kernel(const int64_t* __restrict__ Fin, int L, int len,
                                                                               MeshParams mp, const int64_t* __restrict__ V,
                                                                               uint8_t* __restrict__ bp, size_t bp_stride,
                                                                               int64_t* __restrict__ opt_cost, int32_t* __restrict__ last_sig) {
  using F = Fac<D>;
  using SM = CdpSmem<D>;
  constexpr int K = F::K, ES = F::ES, PARTS = 8, ST = SM::ST;
  constexpr int MAXM = ((D == 3 ? 27 : 9) + PARTS - 1) / PARTS;        // members per thread: the largest valid class has 27 / 9 signatures
  constexpr int NA = (ES + PARTS - 1) / PARTS;
  extern __shared__ __align__(16) unsigned char cdp_raw[];
  SM& sm = *reinterpret_cast<SM*>(cdp_raw);
  const int tid = threadIdx.x, NT = blockDim.x, c = blockIdx.x, C = gridDim.x, p = blockIdx.y;
  const int cls = tid / PARTS, part = tid % PARTS;
  const int t0 = c * len;                                  // the chunk starts from g_{t0}
  const int l_first = c == 0 ? 0 : t0 + 1;                 // first layer whose factors are needed
  const int l_last = (t0 + len + 1 < L - 1 && c + 1 < C) ? t0 + len + 1 : L - 1;
  const int64_t* Fp = Fin + (size_t)p * L * F::FB;
  if (tid == 0) {
    for (int s2 = 0; s2 < ST; ++s2) mbar_init(&sm.full[s2], 1);
    mbar_fence_init();
  }
  __syncthreads();
  const uint64_t pol = policy_evict_first();
  auto fetch = [&](int l) {                                // thread 0
    if (l <= l_last) {
      const int s2 = (l - l_first) % ST;
      mbar_arrive_expect_tx(&sm.full[s2], F::FB * 8);
      bulk_g2s(sm.blk[s2], Fp + (size_t)l * F::FB, F::FB * 8, &sm.full[s2], pol);
    }
  };
  if (tid == 0)
    for (int s2 = 0; s2 < ST; ++s2) fetch(l_first + s2);
  fill_sig_table<D>(sm.sig, mp, tid, NT);
  __syncthreads();
  fill_classes<D>(sm.acls, sm.bcls, sm.sig, tid, NT);
  __syncthreads();
  fill_members<D>(sm.mstart, sm.mlist, sm.acls, tid, NT);
  if (c > 0 && tid < ES) { sm.g[tid] = V[((size_t)p * C + c) * ES + tid]; sm.gi[tid] = 0; }
  __syncthreads();
  bool have_idx = false;                                   // gi holds the smallest index of every class
  uint8_t* bpp = bp + (size_t)p * bp_stride;

  for (int l = l_first; l <= l_last; ++l) {
    mbar_wait(&sm.full[(l - l_first) % ST], ((l - l_first) / ST) & 1);
    const int64_t* blk = sm.blk[(l - l_first) % ST];
    const int kind = (int)blk[0];
    const int64_t* VPl = blk + F::HDR;
    const int64_t* El = blk + F::HDR + K;
    const uint8_t* bc = sm.bcls[kind];
    if (l > 0) {
      // h[b] = min_a g[a] + Esym_l[a][b], the smaller index on ties (an empty class carries 2^61 and never wins)
      int64_t bv = INT64_MAX;
      int bi = 1 << 30;
      if (cls < ES) {
        int64_t v[NA];
        int ix[NA];
#pragma unroll
        for (int q = 0; q < NA; ++q) {
          const int a = part + q * PARTS;
          const bool ok = a < ES;
          v[q] = ok ? sm.g[a] + El[a * ES + cls] : INT64_MAX;
          ix[q] = ok ? sm.gi[a] : 1 << 30;
        }
#pragma unroll
        for (int q = 0; q < NA; ++q)
          if (v[q] < bv || (v[q] == bv && ix[q] < bi)) { bv = v[q]; bi = ix[q]; }
      }
#pragma unroll
      for (int off = 1; off < PARTS; off <<= 1) {          // (every lane of the warp takes part in the shuffles)
        const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
        if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
      }
      if (cls < ES && part == 0) { sm.h[cls] = bv; sm.hi[cls] = bi; }
    } else if (tid < ES) {
      sm.h[tid] = 0;                                       // f_0[j] = T[0][0][j] = VP_0[j]
    }
    __syncthreads();
    if (have_idx)
      for (int j = tid; j < K; j += NT) bpp[(size_t)l * K + j] = (uint8_t)sm.hi[bc[j]];
    // g[a] = min over the signatures j of class a of f_l[j] = VP_l[j] + h[B(j)], smallest j on ties.  The signatures that
    // are invalid for the kind all carry 2^50 and the invalid input class: the first one is the smallest index.
    {
      const uint8_t* ml = sm.mlist[kind];
      int64_t bv = kInfCls;
      int bi = 1 << 30;
      if (cls < ES - 1) {
        const int ms = sm.mstart[kind][cls] + part, m1 = sm.mstart[kind][cls + 1];
        int64_t v[MAXM];
        int ix[MAXM];
#pragma unroll
        for (int q = 0; q < MAXM; ++q) {
          const bool ok = ms + q * PARTS < m1;
          ix[q] = ok ? ml[ms + q * PARTS] : 0;
          v[q] = ok ? VPl[ix[q]] + sm.h[bc[ix[q]]] : kInfCls;
        }
#pragma unroll
        for (int q = 0; q < MAXM; ++q)
          if (v[q] < bv) { bv = v[q]; bi = ix[q]; }
      } else if (cls == ES - 1 && part == 0) {
        const int ms = sm.mstart[kind][ES - 1];
        if (ms < sm.mstart[kind][ES]) { bi = ml[ms]; bv = VPl[bi] + sm.h[ES - 1]; }
      }
#pragma unroll
      for (int off = 1; off < PARTS; off <<= 1) {
        const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
        if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
      }
      if (cls < ES && part == 0) { sm.g[cls] = bv < kInfCls ? bv : kInfCls; sm.gi[cls] = bi; }
    }
    have_idx = true;
    __syncthreads();
    if (tid == 0) fetch(l + ST);                           // the block of layer l has been read by everyone
  }
  if (l_last == L - 1 && tid < 32) {                       // the chain's optimum: smallest argmin of f_{L-1}
    int64_t bv = INT64_MAX;
    int bi = 1 << 30;
    for (int a = tid; a < ES; a += 32)
      if (sm.g[a] < bv || (sm.g[a] == bv && sm.gi[a] < bi)) { bv = sm.g[a]; bi = sm.gi[a]; }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if (tid == 0) { opt_cost[p] = bv; last_sig[p] = bi; }
  }
}

// 5. the walk: strategy[p][l - 1] = bp[p][l][strategy[p][l]]; the chain's back-pointers (bp_stride bytes apart, a 16-byte
// multiple) come to shared memory in one bulk copy when they fit
__global__ void __launch_bounds__(32) chain_walk_kernel(const uint8_t* __restrict__ bp, size_t bp_stride, int L, int K,
                                                        const int32_t* __restrict__ last_sig, int32_t* __restrict__ strategy, int staged) {
  extern __shared__ __align__(128) unsigned char walk_raw[];
  __shared__ uint64_t bar;
  const int p = blockIdx.x, tid = threadIdx.x;
  const uint8_t* bpp = bp + (size_t)p * bp_stride;
  if (tid == 0) {
    const uint8_t* bw = bpp;
    if (staged) {
      mbar_init(&bar, 1);
      mbar_fence_init();
      // (an mbarrier counts at most 2^20 - 1 bytes per phase: pieces of 512 KB at most -- one piece for what fits here)
      mbar_arrive_expect_tx(&bar, (uint32_t)bp_stride);
      bulk_g2s(walk_raw, bpp, (uint32_t)bp_stride, &bar, policy_evict_first());
      mbar_wait(&bar, 0);
      bw = walk_raw;
    }
    int32_t* sp = strategy + (size_t)p * L;
    int sidx = last_sig[p];
    sp[L - 1] = sidx;
    for (int l = L - 1; l >= 1; --l) {
      sidx = bw[(size_t)l * K + sidx];
      sp[l - 1] = sidx;
    }
  }
}

template <int D>
int launch_factors_d(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int64_t* d_F, cudaStream_t st) {
  const int ntiles = Bp * L, sms = device_sm_count();
  const size_t smem = sizeof(FacSmem<D>);
  ADL_CUDA_CHECK(cudaFuncSetAttribute(build_factors_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int per_sm = D == 3 ? 2 : 4;
  const int grid = ntiles < sms * per_sm ? ntiles : sms * per_sm;
  build_factors_kernel<D><<<grid, 256, smem, st>>>(d_layers, ntiles, L, mp, d_F);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

template <int D>
int launch_lookup_d(int32_t Bp, int32_t L, const MeshParams& mp, const int64_t* d_F, uint8_t* d_BR,
                    const int32_t* d_init, int32_t S, int32_t max_sweeps, int64_t* d_cost, int32_t* d_strategy, int32_t* d_sweeps,
                    cudaStream_t st) {
  using F = Fac<D>;
  const int64_t nt64 = (int64_t)Bp * L;
  if (nt64 > 0x7fffffff) { set_error("Bp*L too large"); return AUTODDL_EINVAL; }
  const int ntiles = (int)nt64, sms = device_sm_count();
  {
    const size_t smem = sizeof(BrSmem<D>);
    ADL_CUDA_CHECK(cudaFuncSetAttribute(best_response_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = ntiles < sms * 2 ? ntiles : sms * 2;
    best_response_kernel<D><<<grid, 512, smem, st>>>(d_F, ntiles, L, mp, d_BR);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  {
    const int W = 4;
    const size_t per_warp = ((size_t)2 * 32 * F::CS + 3 * (size_t)L + 15) & ~(size_t)15;
    const size_t shared = (sizeof(SigInfo) * 2 * F::K + 4 * F::K + 15) & ~(size_t)15;
    const size_t smem = shared + W * per_warp;
    if (smem > 200 * 1024) { set_error("coord_descent: L too large"); return AUTODDL_EINVAL; }
    ADL_CUDA_CHECK(cudaFuncSetAttribute(cd_lookup_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t nb = ((int64_t)Bp * S + W - 1) / W;
    if (nb > 0x7fffffff) { set_error("coord_descent: Bp*S too large"); return AUTODDL_EINVAL; }
    cd_lookup_kernel<D><<<(unsigned)nb, W * 32, smem, st>>>(d_F, d_BR, Bp, L, S, mp, d_init, max_sweeps, d_cost, d_strategy, d_sweeps,
                                                            (int)per_warp);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  return AUTODDL_OK;
}

}  // namespace

// layers per chunk: the chunk products and the per-chunk DP grow with it, the serial prefix pass shrinks
static inline int scan_chunk_len(int ndim, int L) { return ndim == 3 && L >= 256 ? 16 : 8; }

template <int D>
int launch_dp_scan_d(const int64_t* d_F, int32_t Bp, int32_t L, const MeshParams& mp, unsigned char* d_work, int64_t* d_opt_cost,
                     int32_t* d_strategy, cudaStream_t st) {
  using F = Fac<D>;
  constexpr int ES = F::ES, N2 = F::N2P, K = F::K;        // (matrices N2P words apart)
  const int len = scan_chunk_len(D, L), C = (L - 2 + len - 1) / len;
  const int sms = device_sm_count();
  // workspace: M [Bp][L][N2P], Q [Bp][C-1][ES][SQ], V [Bp][C][ES] (int64), last signature [Bp] (int32), back-pointers [Bp][bp_stride]
  int64_t* d_M = reinterpret_cast<int64_t*>(d_work);
  int64_t* d_Q = d_M + (size_t)Bp * L * N2;
  int64_t* d_V = d_Q + (size_t)Bp * (C > 1 ? C - 1 : 1) * (ES * F::SQ);
  auto up256 = [](void* q) { return reinterpret_cast<unsigned char*>(((uintptr_t)q + 255) & ~(uintptr_t)255); };
  int32_t* d_last = reinterpret_cast<int32_t*>(up256(d_V + (size_t)Bp * C * ES));
  uint8_t* d_bp = up256(d_last + Bp);                      // (bulk copies want 16-byte aligned sources)
  const int ntiles = Bp * L;
  const size_t bp_stride = ((size_t)L * K + 15) & ~(size_t)15;
  {
    const size_t smem = sizeof(CmSmem<D>);
    ADL_CUDA_CHECK(cudaFuncSetAttribute(class_matrix_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int per_sm = D == 3 ? 2 : 4;
    class_matrix_kernel<D><<<ntiles < sms * per_sm ? ntiles : sms * per_sm, 512, smem, st>>>(d_F, ntiles, mp, d_M);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  if (C > 1) {
    using PC = ProdCfg<D>;
    const size_t smem = ((size_t)2 * N2 + 2 * ES * PC::W) * 8;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(chunk_product_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    chunk_product_kernel<D><<<dim3(C - 1, Bp, PC::NG), PC::NT, smem, st>>>(d_M, L, len, d_Q);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  const int nt8 = (ES * 8 + 31) / 32 * 32;
  {
    const size_t smem = (size_t)4 * ES * F::SQ * 8;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(chunk_prefix_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    chunk_prefix_kernel<D><<<Bp, (ES * 4 + 31) / 32 * 32, smem, st>>>(d_M, L, d_Q, C - 1, d_V);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  {
    const size_t smem = sizeof(CdpSmem<D>);
    ADL_CUDA_CHECK(cudaFuncSetAttribute(chunk_dp_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    chunk_dp_kernel<D><<<dim3(C, Bp), nt8, smem, st>>>(d_F, L, len, mp, d_V, d_bp, bp_stride, d_opt_cost, d_last);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  {
    const int staged = bp_stride <= 200 * 1024;
    const size_t smem = staged ? bp_stride : 16;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(chain_walk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    chain_walk_kernel<<<Bp, 32, smem, st>>>(d_bp, bp_stride, L, K, d_last, d_strategy, staged);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  return AUTODDL_OK;
}

// library-built tables of two or three mesh levels have the factor form these kernels work on
bool factors_supported(const MeshParams& mp) { return (mp.ndim == 2 || mp.ndim == 3) && !mp.fold; }

size_t factors_bytes(const MeshParams& mp, int32_t Bp, int32_t L) {
  const size_t fb = mp.ndim == 2 ? Fac<2>::FB : Fac<3>::FB;
  return ((size_t)Bp * L * fb * 8 + 255) / 256 * 256;
}

int launch_build_factors(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int64_t* d_F, cudaStream_t st) {
  if ((int64_t)Bp * L > 0x7fffffff) { set_error("Bp*L too large"); return AUTODDL_EINVAL; }
  return mp.ndim == 2 ? launch_factors_d<2>(d_layers, Bp, L, mp, d_F, st) : launch_factors_d<3>(d_layers, Bp, L, mp, d_F, st);
}

// many starts per problem: best-response look-ups on the factors
bool cd_lookup_supported(const MeshParams& mp, int32_t L, int32_t S) { return factors_supported(mp) && S >= 32 && L <= 16384; }

// bytes of the best-response tables (the factors are counted by factors_bytes)
size_t cd_lookup_workspace_bytes(const MeshParams& mp, int32_t Bp, int32_t L) {
  const size_t nt = (size_t)Bp * L;
  const size_t es = mp.ndim == 2 ? Fac<2>::ES : Fac<3>::ES, cs = mp.ndim == 2 ? Fac<2>::CS : Fac<3>::CS;
  return (nt * es * cs + 255) / 256 * 256 + 256;
}

int launch_cd_lookup(const int64_t* d_F, int32_t Bp, int32_t L, const MeshParams& mp, void* d_work, const int32_t* d_init, int32_t S,
                     int32_t max_sweeps, int64_t* d_cost, int32_t* d_strategy, int32_t* d_sweeps, cudaStream_t st) {
  uint8_t* d_BR = (uint8_t*)d_work;
  if (mp.ndim == 2) return launch_lookup_d<2>(Bp, L, mp, d_F, d_BR, d_init, S, max_sweeps, d_cost, d_strategy, d_sweeps, st);
  return launch_lookup_d<3>(Bp, L, mp, d_F, d_BR, d_init, S, max_sweeps, d_cost, d_strategy, d_sweeps, st);
}

// chain DP of few long chains, parallel over the layers (on the factors): two / three mesh levels, L >= 32, Bp <= 64
bool chain_dp_scan_supported(const MeshParams& mp, int32_t Bp, int32_t L) { return factors_supported(mp) && L >= 32 && Bp <= 64; }

size_t chain_dp_scan_bytes(const MeshParams& mp, int32_t Bp, int32_t L) {
  const int es = mp.ndim == 2 ? Fac<2>::ES : Fac<3>::ES, k = mp.ndim == 2 ? Fac<2>::K : Fac<3>::K, len = scan_chunk_len(mp.ndim, L);
  const size_t n2 = mp.ndim == 2 ? Fac<2>::N2P : Fac<3>::N2P, c = (L - 2 + len - 1) / len;
  const size_t qw = (size_t)es * (mp.ndim == 2 ? Fac<2>::SQ : Fac<3>::SQ);
  const size_t b = ((size_t)Bp * L * n2 + (size_t)Bp * (c > 1 ? c - 1 : 1) * qw + (size_t)Bp * c * es) * 8 +
                   (((size_t)Bp * 4 + 255) & ~(size_t)255) + (size_t)Bp * (((size_t)L * k + 15) & ~(size_t)15);
  return (b + 255) / 256 * 256 + 768;                      // (+ the alignment gaps of the carve-up)
}

int launch_chain_dp_scan(const int64_t* d_F, int32_t Bp, int32_t L, const MeshParams& mp, void* d_work, int64_t* d_opt_cost,
                         int32_t* d_strategy, cudaStream_t st) {
  return mp.ndim == 2 ? launch_dp_scan_d<2>(d_F, Bp, L, mp, (unsigned char*)d_work, d_opt_cost, d_strategy, st)
                      : launch_dp_scan_d<3>(d_F, Bp, L, mp, (unsigned char*)d_work, d_opt_cost, d_strategy, st);
}

}  // namespace autoddl
