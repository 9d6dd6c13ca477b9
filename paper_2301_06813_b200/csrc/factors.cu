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
#include "factors.cuh"

namespace autoddl {

namespace {

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
  fill_members<D>(sm.mstart, sm.mlist, sm.acls, tid, NT);   // the candidates of every producer class, ascending
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

// ---- the same look-up scheme on K x K TABLES, K <= 64 (caller-supplied tables, meshes without the factor form) -----------
// Without classes the neighbours enter the update of layer l as themselves: BRt[l][j'][i] = smallest-index argmin_c
// T[l][i][c] + T[l+1][c][j']  (K^3 operations per layer; layer 0's row is T[0][0][.], the last layer has no right term and
// only its column 0 is used).  The 16-bit entry is (c, c), so the walk below is the walk of cd_lookup_kernel.
__global__ void __launch_bounds__(512) best_response_tab_kernel(const int64_t* __restrict__ T, int ntiles, int L, int K, int CS,
                                                                uint8_t* __restrict__ BRt) {
  constexpr int NT = 512;
  extern __shared__ __align__(16) unsigned char brt_raw[];
  const int n = K * K, tid = threadIdx.x;
  int64_t* Tl = reinterpret_cast<int64_t*>(brt_raw);
  int64_t* Tr = Tl + n;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int l = tile % L;
    const bool has_right = l < L - 1;
    const int64_t* tl = T + (size_t)tile * n;
    __syncthreads();
    for (int x = tid; x < n; x += NT) {
      Tl[x] = __ldg(tl + (l == 0 ? x % K : x));            // (layer 0: every row is row 0, s_{-1} := 0)
      Tr[x] = has_right ? __ldg(tl + n + x) : 0;
    }
    __syncthreads();
    uint8_t* out = BRt + (size_t)tile * K * CS;
    const int ncol = has_right ? K : 1;
    for (int o = tid; o < K * ncol; o += NT) {
      const int i = o / ncol, jr = o % ncol;
      const int64_t* a = Tl + i * K;
      const int64_t* b = Tr + jr;
      int64_t best = INT64_MAX;
      int arg = 0;
      for (int c = 0; c < K; ++c) {
        const int64_t g = a[c] + b[c * K];
        if (g < best) { best = g; arg = c; }               // increasing c, strict '<': the smallest index
      }
      reinterpret_cast<uint16_t*>(out + (size_t)jr * CS)[i] = (uint16_t)(arg | arg << 8);
    }
  }
}

__global__ void __launch_bounds__(128) cd_lookup_tab_kernel(const int64_t* __restrict__ T, const uint8_t* __restrict__ BRt, int Bp, int L,
                                                            int K, int CS, int S, const int32_t* __restrict__ init, int max_sweeps,
                                                            int64_t* __restrict__ cost, int32_t* __restrict__ strategy,
                                                            int32_t* __restrict__ sweeps, int per_warp_bytes) {
  extern __shared__ __align__(16) unsigned char cdt_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, W = blockDim.x >> 5;
  const size_t ps = (size_t)blockIdx.x * W + warp;
  if (ps >= (size_t)Bp * S) return;
  const size_t p = ps / S;
  unsigned char* wb = cdt_raw + (size_t)warp * per_warp_bytes;
  uint8_t* chunk = wb;                                     // [2][32][CS] best-response columns of 32 layers, double buffered
  uint8_t* s = chunk + 2 * 32 * CS;                        // [L] strategy
  uint8_t* dirty = s + L;                                  // [L]
  const uint8_t* Bp_ = BRt + p * (size_t)L * K * CS;
  for (int l = lane; l < L; l += 32) {
    s[l] = (uint8_t)init[ps * L + l];
    dirty[l] = 1;
  }
  __syncwarp();
  // column of layer l for the CURRENT right neighbour (old s_{l+1}: it is not touched before layer l + 1's own turn)
  auto fetch = [&](int l0, int b) {                        // lane i -> layer l0 + i -> chunk[b][i][0 .. CS), asynchronously
    const int l = l0 + lane;
    if (l < L) {
      const int right = l < L - 1 ? s[l + 1] : 0;
      const unsigned char* src = Bp_ + ((size_t)l * K + right) * CS;
      unsigned char* dst = chunk + ((size_t)b * 32 + lane) * CS;
      for (int q = 0; q < CS / 16; ++q) cp_async16(dst + 16 * q, src + 16 * q);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  int nsweeps = 0;
  for (;;) {                                               // (the sweep of cd_lookup_kernel with identity classes)
    bool changed = false, carry = false, have = false;
    int aprev = 0, cb = 0;
    for (int l0 = 0; l0 < L; l0 += 32) {
      const int n = L - l0 < 32 ? L - l0 : 32;
      int sreg = lane < n ? s[l0 + lane] : 0;
      const unsigned dmask = __ballot_sync(0xffffffffu, lane < n && dirty[l0 + lane]);
      if (dmask == 0 && !carry) {
        aprev = __shfl_sync(0xffffffffu, sreg, n - 1);
        if (have) asm volatile("cp.async.wait_group 0;" ::: "memory");
        have = false;
        continue;
      }
      if (!have) fetch(l0, cb);
      const bool ahead = l0 + 32 < L;
      if (ahead) fetch(l0 + 32, cb ^ 1);
      if (ahead) asm volatile("cp.async.wait_group 1;" ::: "memory"); else asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncwarp();
      const uint16_t* colb = reinterpret_cast<const uint16_t*>(chunk + (size_t)cb * 32 * CS);
      const int i0 = carry ? 0 : __ffs(dmask) - 1;
      if (i0 > 0) aprev = __shfl_sync(0xffffffffu, sreg, i0 - 1);
      int mine = sreg;
      for (int i = i0; i < n; ++i) {
        const int e = colb[i * (CS / 2) + aprev] & 255;
        if (lane == i) mine = e;
        aprev = e;
      }
      const unsigned chm = __ballot_sync(0xffffffffu, lane < n && mine != sreg);
      if (chm) changed = true;
      carry = chm >> (n - 1) & 1;
      const unsigned dnext = chm >> 1;
      if ((chm & 1) && l0 > 0 && lane == 0) dirty[l0 - 1] = 1;
      sreg = mine;
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
  const int64_t* Tp = T + p * (size_t)L * K * K;           // Cost(s) = sum_l T[l][s_{l-1}][s_l]   (s_{-1} := 0)
  int64_t acc = 0;
  for (int l = lane; l < L; l += 32) {
    const int sl = s[l], sp = l > 0 ? s[l - 1] : 0;
    acc += __ldg(Tp + ((size_t)l * K + sp) * K + sl);
    strategy[ps * L + l] = sl;
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
  if (lane == 0) {
    cost[ps] = acc;
    sweeps[ps] = nsweeps;
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

// best-response look-ups on K x K tables: any mesh, K <= 64, >= 32 starts per problem
bool cd_lookup_tab_supported(int32_t K, int32_t L, int32_t S) { return K <= 64 && S >= 32 && L <= 16384; }

static inline size_t tab_cs(int32_t K) { return ((size_t)2 * K + 15) / 16 * 16; }

size_t cd_lookup_tab_workspace_bytes(int32_t K, int32_t Bp, int32_t L) { return ((size_t)Bp * L * K * tab_cs(K) + 255) / 256 * 256 + 256; }

int launch_cd_lookup_tab(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, void* d_work, const int32_t* d_init, int32_t S,
                         int32_t max_sweeps, int64_t* d_cost, int32_t* d_strategy, int32_t* d_sweeps, cudaStream_t st) {
  uint8_t* d_BR = (uint8_t*)d_work;
  const int CS = (int)tab_cs(K);
  const int64_t nt64 = (int64_t)Bp * L;
  if (nt64 > 0x7fffffff) { set_error("Bp*L too large"); return AUTODDL_EINVAL; }
  const int ntiles = (int)nt64, sms = device_sm_count();
  {
    const size_t smem = (size_t)2 * K * K * 8;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(best_response_tab_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = ntiles < sms * 2 ? ntiles : sms * 2;
    best_response_tab_kernel<<<grid, 512, smem, st>>>(d_T, ntiles, L, K, CS, d_BR);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  {
    const int W = 4;
    const size_t per_warp = ((size_t)2 * 32 * CS + 2 * (size_t)L + 15) & ~(size_t)15;
    const size_t smem = W * per_warp;
    if (smem > 200 * 1024) { set_error("coord_descent: L too large"); return AUTODDL_EINVAL; }
    ADL_CUDA_CHECK(cudaFuncSetAttribute(cd_lookup_tab_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t nb = ((int64_t)Bp * S + W - 1) / W;
    if (nb > 0x7fffffff) { set_error("coord_descent: Bp*S too large"); return AUTODDL_EINVAL; }
    cd_lookup_tab_kernel<<<(unsigned)nb, W * 32, smem, st>>>(d_T, d_BR, Bp, L, K, CS, S, d_init, max_sweeps, d_cost, d_strategy, d_sweeps,
                                                             (int)per_warp);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  return AUTODDL_OK;
}

}  // namespace autoddl
