// Chain DP (R9) of few long chains, parallel over the layers, on the factors of the cost tables.
#include "factors.cuh"

namespace autoddl {

namespace {

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

// ---- the same scheme on K x K TABLES (caller-supplied, or built for a mesh without the factor form), K <= 64 -------------
// Without classes the state is f_l itself and the matrices are the tiles: Q_c = T_{t_c+1} (x) ... (x) T_{t_c+len}, V_0 = f_0 =
// T[0][0][.], V_{c+1} = V_c (x) Q_c = f_{t_{c+1}}, and the CTA of chunk c runs the ordinary DP over layers t_c+1 .. t_c+len
// from f_{t_c} (smallest i on ties: the sequential DP on its chunk).  K^3 <= 2.6e5 operations per product: a CTA per chunk.
__device__ __forceinline__ void cp_async8(void* dst_smem, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// one K x K tile global -> shared by all threads of the CTA (tiles of an odd K are only 8-byte aligned); one commit group
__device__ __forceinline__ void tile_g2s(int64_t* dst, const int64_t* src, int K, int tid, int nt) {
  const int n = K * K;
  if ((K & 1) == 0)
    for (int x = tid; x < n / 2; x += nt) cp_async16(dst + 2 * x, src + 2 * x);
  else
    for (int x = tid; x < n; x += nt) cp_async8(dst + x, src + x);
  cp_async_commit();
}

// Q[p][c] = T_{t_c + 1} (x) ... (x) T_{t_c + len} for c = 0 .. C - 2 (grid.x = C - 1, grid.y = Bp); matrices QS words apart
__global__ void __launch_bounds__(512) chunk_product_tab_kernel(const int64_t* __restrict__ T, int L, int K, int len,
                                                                int64_t* __restrict__ Q, int QS) {
  constexpr int NT = 512, MAXO = 8;                        // outputs per thread: 64 x 64 / 512
  extern __shared__ __align__(128) unsigned char tp_raw[];
  const int n = K * K, nb = (n + 1) & ~1;
  int64_t* A = reinterpret_cast<int64_t*>(tp_raw);
  int64_t* Bb = A + nb;
  const int tid = threadIdx.x, c = blockIdx.x, p = blockIdx.y;
  const int64_t* T1 = T + ((size_t)p * L + (size_t)c * len + 1) * n;       // T_{t_c + 1}
  tile_g2s(A, T1, K, tid, NT);
  if (len > 1) tile_g2s(Bb + nb, T1 + n, K, tid, NT);      // T_{t_c + 1 + k} -> buffer k & 1
  for (int k = 1; k < len; ++k) {
    if (k + 1 < len) { tile_g2s(Bb + ((k + 1) & 1) * nb, T1 + (size_t)(k + 1) * n, K, tid, NT); cp_async_wait_group<1>(); }
    else cp_async_wait_group<0>();
    __syncthreads();
    const int64_t* B = Bb + (k & 1) * nb;
    int64_t best[MAXO];
#pragma unroll
    for (int q = 0; q < MAXO; ++q) {
      const int o = tid + q * NT;
      best[q] = INT64_MAX;
      if (o < n) {
        const int64_t* a = A + o / K * K;
        const int64_t* b = B + o % K;
        int64_t bv = INT64_MAX;
        for (int m = 0; m < K; ++m) {
          const int64_t g = a[m] + b[m * K];
          bv = g < bv ? g : bv;
        }
        best[q] = bv;
      }
    }
    __syncthreads();                                       // A and the buffer have been read by everyone
#pragma unroll
    for (int q = 0; q < MAXO; ++q)
      if (tid + q * NT < n) A[tid + q * NT] = best[q];
  }
  if (len == 1) cp_async_wait_group<0>();
  __syncthreads();
  int64_t* out = Q + ((size_t)p * gridDim.x + c) * QS;
  for (int x = tid; x < n; x += NT) out[x] = A[x];
}

// V[p][0] = f_0 = T[p][0][0][.], V[p][c + 1] = V[p][c] (x) Q[p][c]   (one CTA per chain, 4 threads per output, TMA ring)
__global__ void __launch_bounds__(256) chunk_prefix_tab_kernel(const int64_t* __restrict__ T, int L, int K, const int64_t* __restrict__ Q,
                                                               int QS, int nq, int64_t* __restrict__ V) {
  constexpr int PARTS = 4, ST = 4;
  extern __shared__ __align__(128) unsigned char tf_raw[];
  int64_t* ring = reinterpret_cast<int64_t*>(tf_raw);      // ST matrices
  __shared__ int64_t v[2][64];
  __shared__ uint64_t full[ST];
  const int tid = threadIdx.x, p = blockIdx.x;
  const int b = tid / PARTS, part = tid % PARTS;
  const int64_t* Qp = Q + (size_t)p * nq * QS;
  if (tid == 0) {
    for (int s2 = 0; s2 < ST; ++s2) mbar_init(&full[s2], 1);
    mbar_fence_init();
  }
  __syncthreads();
  const uint64_t pol = policy_evict_first();
  auto fetch = [&](int c) {                                // thread 0
    if (c < nq) {
      mbar_arrive_expect_tx(&full[c % ST], QS * 8);
      bulk_g2s(ring + (size_t)(c % ST) * QS, Qp + (size_t)c * QS, QS * 8, &full[c % ST], pol);
    }
  };
  if (tid == 0)
    for (int s2 = 0; s2 < ST; ++s2) fetch(s2);
  if (tid < K) {
    const int64_t f0 = T[(size_t)p * L * K * K + tid];
    v[0][tid] = f0;
    V[(size_t)p * (nq + 1) * K + tid] = f0;
  }
  __syncthreads();
  for (int c = 0; c < nq; ++c) {
    mbar_wait(&full[c % ST], (c / ST) & 1);
    const int64_t* Qc = ring + (size_t)(c % ST) * QS + (b < K ? b : 0);
    const int64_t* vin = v[c & 1];
    int64_t best = INT64_MAX;
    for (int a = part; a < K; a += PARTS) {
      const int64_t g = vin[a] + Qc[a * K];
      best = g < best ? g : best;
    }
#pragma unroll
    for (int off = 1; off < PARTS; off <<= 1) {
      const int64_t o = __shfl_xor_sync(0xffffffffu, best, off);
      best = o < best ? o : best;
    }
    if (b < K && part == 0) {
      v[(c & 1) ^ 1][b] = best;
      V[((size_t)p * (nq + 1) + c + 1) * K + b] = best;
    }
    __syncthreads();
    if (tid == 0) fetch(c + ST);
  }
}

// the DP of chunk c of chain p over layers t_c + 1 .. min(t_c + len, L - 1), from V[p][c] = f_{t_c} (grid.x = C, grid.y = Bp)
__global__ void __launch_bounds__(512) chunk_dp_tab_kernel(const int64_t* __restrict__ T, int L, int K, int len,
                                                           const int64_t* __restrict__ V, uint8_t* __restrict__ bp, size_t bp_stride,
                                                           int64_t* __restrict__ opt_cost, int32_t* __restrict__ last_sig) {
  constexpr int NT = 512, PARTS = 8;
  extern __shared__ __align__(128) unsigned char td_raw[];
  const int n = K * K, nb = (n + 1) & ~1;
  int64_t* tiles = reinterpret_cast<int64_t*>(td_raw);     // two buffers
  __shared__ int64_t f[64];
  const int tid = threadIdx.x, c = blockIdx.x, C = gridDim.x, p = blockIdx.y;
  const int j = tid / PARTS, part = tid % PARTS;
  const int l0 = c * len + 1, l1 = (l0 + len - 1 < L - 1 && c + 1 < C) ? l0 + len - 1 : L - 1;
  const int64_t* Tp = T + (size_t)p * L * n;
  uint8_t* bpp = bp + (size_t)p * bp_stride;
  tile_g2s(tiles, Tp + (size_t)l0 * n, K, tid, NT);
  if (tid < K) f[tid] = V[((size_t)p * C + c) * K + tid];
  for (int l = l0; l <= l1; ++l) {
    if (l + 1 <= l1) { tile_g2s(tiles + ((l + 1 - l0) & 1) * nb, Tp + (size_t)(l + 1) * n, K, tid, NT); cp_async_wait_group<1>(); }
    else cp_async_wait_group<0>();
    __syncthreads();
    const int64_t* tl = tiles + ((l - l0) & 1) * nb + (j < K ? j : 0);
    int64_t bv = INT64_MAX;
    int bi = 1 << 30;
    if (j < K)
      for (int i = part; i < K; i += PARTS) {              // increasing i and strict '<': the thread keeps its smallest i
        const int64_t g = f[i] + tl[i * K];
        if (g < bv) { bv = g; bi = i; }
      }
#pragma unroll
    for (int off = 1; off < PARTS; off <<= 1) {
      const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    __syncthreads();                                       // f_{l-1} and the tile have been read by everyone
    if (j < K && part == 0) {
      f[j] = bv;
      bpp[(size_t)l * K + j] = (uint8_t)bi;
    }
  }
  __syncthreads();
  if (l1 == L - 1 && tid < 32) {                           // the chain's optimum: smallest argmin of f_{L-1}
    int64_t bv = INT64_MAX;
    int bi = 1 << 30;
    for (int a = tid; a < K; a += 32)
      if (f[a] < bv) { bv = f[a]; bi = a; }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if (tid == 0) { opt_cost[p] = bv; last_sig[p] = bi; }
  }
}

constexpr int kTabScanLen = 8, kTabScanMaxK = 64;

int launch_dp_scan_tab(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, unsigned char* d_work, int64_t* d_opt_cost,
                       int32_t* d_strategy, cudaStream_t st) {
  const int len = kTabScanLen, C = (L - 1 + len - 1) / len, n = K * K, QS = (n + 1) & ~1;
  // workspace: Q [Bp][C-1][QS], V [Bp][C][K] (int64), last signature [Bp] (int32), back-pointers [Bp][bp_stride]
  auto up256 = [](void* q) { return reinterpret_cast<unsigned char*>(((uintptr_t)q + 255) & ~(uintptr_t)255); };
  int64_t* d_Q = reinterpret_cast<int64_t*>(d_work);
  int64_t* d_V = d_Q + (size_t)Bp * (C > 1 ? C - 1 : 1) * QS;
  int32_t* d_last = reinterpret_cast<int32_t*>(up256(d_V + (size_t)Bp * C * K));
  uint8_t* d_bp = up256(d_last + Bp);
  const size_t bp_stride = ((size_t)L * K + 15) & ~(size_t)15;
  if (C > 1) {
    const size_t smem = (size_t)3 * QS * 8;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(chunk_product_tab_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    chunk_product_tab_kernel<<<dim3(C - 1, Bp), 512, smem, st>>>(d_T, L, K, len, d_Q, QS);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  {
    const size_t smem = (size_t)4 * QS * 8;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(chunk_prefix_tab_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    chunk_prefix_tab_kernel<<<Bp, 256, smem, st>>>(d_T, L, K, d_Q, QS, C - 1, d_V);
    count_launch();
    ADL_CUDA_CHECK(cudaGetLastError());
  }
  {
    const size_t smem = (size_t)2 * QS * 8;
    ADL_CUDA_CHECK(cudaFuncSetAttribute(chunk_dp_tab_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    chunk_dp_tab_kernel<<<dim3(C, Bp), 512, smem, st>>>(d_T, L, K, len, d_V, d_bp, bp_stride, d_opt_cost, d_last);
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

}  // namespace

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


// the same on K x K tables: any mesh, K <= 64, L >= 32, Bp <= 64
bool chain_dp_scan_tab_supported(int32_t K, int32_t Bp, int32_t L) { return K <= kTabScanMaxK && L >= 32 && Bp <= 64; }

size_t chain_dp_scan_tab_bytes(int32_t K, int32_t Bp, int32_t L) {
  const size_t c = (L - 1 + kTabScanLen - 1) / kTabScanLen, qs = ((size_t)K * K + 1) & ~(size_t)1;
  const size_t b = ((size_t)Bp * (c > 1 ? c - 1 : 1) * qs + (size_t)Bp * c * K) * 8 + (((size_t)Bp * 4 + 255) & ~(size_t)255) +
                   (size_t)Bp * (((size_t)L * K + 15) & ~(size_t)15);
  return (b + 255) / 256 * 256 + 768;
}

int launch_chain_dp_scan_tab(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, void* d_work, int64_t* d_opt_cost,
                             int32_t* d_strategy, cudaStream_t st) {
  return launch_dp_scan_tab(d_T, Bp, L, K, (unsigned char*)d_work, d_opt_cost, d_strategy, st);
}
}  // namespace autoddl

// ---- autoddl_chain_dp_static: the layer-parallel chain DP on K x K tables with its scratch in a STATIC device array ----------
// For callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc):
// the chunk products Q, the prefix vectors V, the last signatures and the back-pointers of launch_dp_scan_tab live in a
// file-scope array of AUTODDL_STATIC_SCRATCH_BYTES; every GPU that loads the library holds it until exit.  In host code
// the array's name is a host-side stand-in, not a device address: the address comes from cudaGetSymbolAddress, once per
// device, with that device current.  No cudaMalloc / cudaFree / allocating library routine is called here or in the
// launcher.  Nothing has to start at zero: every word a kernel of the call reads was written by an earlier kernel of the same
// call (the array keeps the last call's contents; tests poison it).  All calls share the array: calls that overlap on the
// GPU (two streams, two host threads) race.
namespace autoddl {
namespace {

static __device__ __align__(256) unsigned char g_static_scratch[AUTODDL_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
void* g_static_ptr[kMaxDevices];                           // device address of g_static_scratch per device (NULL: not asked yet)

// device address of the array on the CURRENT device; AUTODDL_OK or AUTODDL_ECUDA
int static_scratch_address(void** out) {
  int dev = -1;
  ADL_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) { set_error("chain_dp_static: device %d out of range", dev); return AUTODDL_ECUDA; }
  void* p = __atomic_load_n(&g_static_ptr[dev], __ATOMIC_ACQUIRE);
  if (p == nullptr) {
    ADL_CUDA_CHECK(cudaGetSymbolAddress(&p, g_static_scratch));      // (the same value whichever thread asks first)
    if (p == nullptr) { set_error("chain_dp_static: cudaGetSymbolAddress returned NULL"); return AUTODDL_ECUDA; }
    __atomic_store_n(&g_static_ptr[dev], p, __ATOMIC_RELEASE);
  }
  *out = p;
  return AUTODDL_OK;
}

}  // namespace
}  // namespace autoddl

extern "C" {

size_t autoddl_chain_dp_static_bytes(int32_t Bp, int32_t L, const autoddl_mesh* mesh) {
  using namespace autoddl;
  clear_error();
  MeshParams mp;
  if (validate_mesh_net(mesh, nullptr, &mp) || Bp < 1 || L < 1) return 0;
  if (!chain_dp_scan_tab_supported(mp.K, Bp, L)) return 0;
  return chain_dp_scan_tab_bytes(mp.K, Bp, L);
}

int autoddl_chain_dp_static(const int64_t* d_T, int32_t Bp, int32_t L, const autoddl_mesh* mesh, int64_t* d_opt_cost,
                            int32_t* d_strategy, void* stream) {
  using namespace autoddl;
  clear_error();
  MeshParams mp;
  int rc = validate_mesh_net(mesh, nullptr, &mp);
  if (rc) return rc;
  ADL_REQUIRE(d_T != nullptr && d_opt_cost != nullptr && d_strategy != nullptr, "NULL pointer");
  ADL_REQUIRE(((uintptr_t)d_T & 7) == 0 && ((uintptr_t)d_opt_cost & 7) == 0 && ((uintptr_t)d_strategy & 3) == 0, "misaligned pointer");
  ADL_REQUIRE(Bp >= 1 && L >= 1, "Bp = %d, L = %d must be >= 1", Bp, L);
  const int K = mp.K;
  ADL_REQUIRE(chain_dp_scan_tab_supported(K, Bp, L),
              "chain_dp_static: K = %d, Bp = %d, L = %d outside K <= 64, Bp <= 64, L >= 32 (use autoddl_chain_dp)", K, Bp, L);
  const size_t need = chain_dp_scan_tab_bytes(K, Bp, L);
  if (need > (size_t)AUTODDL_STATIC_SCRATCH_BYTES) {
    set_error("chain_dp_static: %zu bytes of scratch needed, the static array holds %zu (use autoddl_chain_dp with a workspace)",
              need, (size_t)AUTODDL_STATIC_SCRATCH_BYTES);
    return AUTODDL_EWORK;
  }
  void* scratch = nullptr;
  if ((rc = static_scratch_address(&scratch))) return rc;
  return launch_chain_dp_scan_tab(d_T, Bp, L, K, scratch, d_opt_cost, d_strategy, (cudaStream_t)stream);
}

}  // extern "C"
