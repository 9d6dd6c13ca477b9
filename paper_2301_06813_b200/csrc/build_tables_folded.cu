// (a1) for the FOLDED factorisation space (R28; PAPER.md:193 p = p0 p1 p2, :201 (nodes, GPUs) tuples): up to
// eight mesh levels, one signature per ordered factorisation of every group of equal levels (K <= 256; 28 / 36 / 45 on
// 2^6 / 2^7 / 2^8 single-GPU nodes).  The 3^D split-configuration tables of the other builders do not exist at D = 8,
// so a cell walks its redistribution itself -- but on bit masks: a tensor state is (m0, m1) = the sets of levels that
// split its rows / columns, the local size is Q_rows[m0] * Q_cols[m1] with Q[x][m] = ceil(extent x / product of the levels
// in m) tabulated once per tile for all 2^D subsets (no division in the walk), and a level's state is two bits of a
// packed word.  One CTA per tile (grid-stride), one thread per cell.
#include "sbp_builder.cuh"

namespace autoddl {

namespace {

constexpr int kFoldNT = 256;

struct FoldSmem {
  int64_t Q[5][256];                                     // M, Kd, N, in_rows, in_cols  x  level subset
  int64_t VP[256];
  uint16_t dig[256];                                     // per signature: row (0, 1, 2) of level d at bits 2d
  // per (layer kind, signature), once per CTA: the level sets (fold_sets) of the output states, the input states and their
  // duals; ok = valid for the kind
  uint32_t stO[2][256], stI[2][256], duO[2][256], duI[2][256];
  uint8_t ok[2][256];
  // the levels' parameters: per-thread indices into the kernel parameters (constant bank) would serialise
  int64_t lv_alpha[8], lv_beta[8], lv_size[8];
  uint64_t lv_magic[8];
  RecBuf rec;
};

// packed per-level states (two bits per level) of a signature's digits for a layer kind; false if invalid for the kind
__device__ __forceinline__ bool fold_states(int kind, uint32_t dig, int D, uint32_t& sI, uint32_t& sW, uint32_t& sO) {
  sI = sW = sO = 0;
  bool valid = true;
  for (int d = 0; d < D; ++d) {
    const int g = dig >> (2 * d) & 3;
    int i, w, o;
    if (kind == AUTODDL_GEMM) { i = c_gemm_I[g]; w = c_gemm_W[g]; o = c_gemm_O[g]; }
    else { i = o = c_attn_IO[g]; w = kB; if (i < 0) { valid = false; i = o = kB; } }
    sI |= i << (2 * d); sW |= w << (2 * d); sO |= o << (2 * d);
  }
  return valid;
}

// level sets of a packed state word (two bits per level): S0 | S1 << 8 | B << 16 | P << 24
__device__ __forceinline__ uint32_t fold_sets(uint32_t s, int D) {
  uint32_t r = 0;
  for (int d = 0; d < D; ++d) r |= 1u << (8 * (s >> (2 * d) & 3) + d);
  return r;
}
__device__ __forceinline__ uint32_t fold_sets_dual(uint32_t m) { return (m & 0xffffu) | (m >> 8 & 0xff0000u) | (m << 8 & 0xff000000u); }   // B <-> P

// forward redistribution a -> b of the layer's input tensor (R4): slice, reduce-scatter (innermost level
// first, message = tensor before), all-to-all (innermost first, message = tensor after), all-gather (outermost first,
// message = tensor after); Table 2 with the level's size and link parameters.  a, b: level sets
// (fold_sets).  Which levels run which collective follows from the sets alone (a level's state only changes at its own
// turn), so each phase visits only the levels that do something; the message sizes use the running split masks.
__device__ int64_t fold_walk(uint32_t a, uint32_t b, const int64_t* __restrict__ Qr, const int64_t* __restrict__ Qc,
                             int64_t eb, const FoldSmem& lv) {
  const uint32_t tS0 = b & 255, tS1 = b >> 8 & 255, tB = b >> 16 & 255, tP = b >> 24;
  const uint32_t aB = a >> 16 & 255;
  uint32_t m0 = (a & 255) | (aB & tS0), m1 = (a >> 8 & 255) | (aB & tS1);      // replicated -> split: keep the own slice, free
  int64_t cost = 0;
  for (uint32_t r = (a >> 24) & ~tP; r;) {               // partial sums: reduce-scatter, innermost level first
    const int d = 31 - __clz(r);
    r ^= 1u << d;
    const int64_t n = Qr[m0] * Qc[m1] * eb, p = lv.lv_size[d];
    if (p > 1) cost += (p - 1) * (lv.lv_alpha[d] + cdiv_magic(n, (uint32_t)p, lv.lv_magic[d]) * lv.lv_beta[d]);
    if (tS0 >> d & 1) m0 |= 1u << d; else m1 |= 1u << d;   // P -> B scatters on axis 1 and gathers later
  }
  for (uint32_t x = (m0 & tS1) | (m1 & tS0); x;) {       // change of split axis: all-to-all, innermost first
    const int d = 31 - __clz(x);
    x ^= 1u << d;
    m0 ^= 1u << d; m1 ^= 1u << d;
    const int64_t n = Qr[m0] * Qc[m1] * eb, p = lv.lv_size[d];
    if (p > 1) cost += (p - 1) * lv.lv_alpha[d] + n * lv.lv_beta[d];
  }
  for (uint32_t g = (m0 | m1) & tB; g;) {                // split -> replicated: all-gather, outermost first
    const int d = __ffs(g) - 1;
    g ^= 1u << d;
    m0 &= ~(1u << d); m1 &= ~(1u << d);
    const int64_t n = Qr[m0] * Qc[m1] * eb, p = lv.lv_size[d];
    if (p > 1) cost += (p - 1) * (lv.lv_alpha[d] + cdiv_magic(n, (uint32_t)p, lv.lv_magic[d]) * lv.lv_beta[d]);
  }
  return cost;                                           // (-> P is a zero fill, free)
}

__global__ void __launch_bounds__(kFoldNT) build_tables_folded_kernel(const autoddl_layer* __restrict__ layers, int ntiles, int L,
                                                                      int chunks, MeshParams mp, int64_t* __restrict__ T,
                                                                      int64_t* __restrict__ node, uint8_t* __restrict__ mask) {
  __shared__ FoldSmem sm;
  const int tid = threadIdx.x, D = mp.ndim, K = mp.K;
  // signature index -> digits: mixed radix over the groups (group 0 most significant); inside a group of n levels the
  // x-th sorted string 0^n0 1^n1 2^n2 in increasing lexicographic order (n0 descending, then n1 descending)
  for (int j = tid; j < K; j += kFoldNT) {
    uint32_t dg = 0;
    int r = j;
    for (int g = mp.ngroups - 1; g >= 0; --g) {
      const int n = mp.glen[g], radix = (n + 2) * (n + 1) / 2;
      int x = r % radix;
      r /= radix;
      int n0 = n, n1 = 0;
      while (x > n - n0) { x -= n - n0 + 1; --n0; }      // n0 = n has 1 string, n0 = n - 1 has 2, ...
      n1 = n - n0 - x;
      for (int t = 0; t < n; ++t) dg |= (uint32_t)(t < n0 ? 0 : (t < n0 + n1 ? 1 : 2)) << (2 * (mp.gfirst[g] + t));
    }
    sm.dig[j] = (uint16_t)dg;
  }
  __syncthreads();
  for (int x = tid; x < 2 * K; x += kFoldNT) {
    const int kind = x / K, j = x % K;
    uint32_t sI, sW, sO;
    const bool valid = fold_states(kind, sm.dig[j], D, sI, sW, sO);
    sm.stO[kind][j] = fold_sets(sO, D);
    sm.stI[kind][j] = fold_sets(sI, D);
    sm.duO[kind][j] = fold_sets_dual(sm.stO[kind][j]);
    sm.duI[kind][j] = fold_sets_dual(sm.stI[kind][j]);
    sm.ok[kind][j] = valid;
  }
  if (tid < 8) {
    sm.lv_size[tid] = tid < D ? mp.size[tid] : 1;
    sm.lv_alpha[tid] = tid < D ? mp.alpha[tid] : 0;
    sm.lv_beta[tid] = tid < D ? mp.beta[tid] : 0;
    sm.lv_magic[tid] = tid < D ? mp.magic_size[tid] : 0;
  }
  const int64_t cap_layer = mp.mem_cap / L;

  // a unit = (tile, chunk of its cells): few tiles (one model) are split so that every SM holds several CTAs -- the walk of
  // a cell is a long dependent chain, and occupancy is what hides it; Q and VP are recomputed per unit (cheap next to the cells)
  for (int unit = blockIdx.x; unit < ntiles * chunks; unit += gridDim.x) {
    const int tile = unit / chunks, chunk = unit % chunks;
    const int l = tile % L;
    __syncthreads();                                     // the previous tile's readers are done
    if (tid == 0) {
      const autoddl_layer* cur = layers + tile;
      RecBuf& r = sm.rec;
      r.X[0] = cur->M; r.X[1] = cur->Kd; r.X[2] = cur->N; r.X[3] = cur->in_rows; r.X[4] = cur->in_cols;
      r.kind = cur->kind; r.eb = cur->act_bytes; r.wgb = cur->wgrad_bytes; r.wsb = cur->wstate_bytes;
      r.maxr = cur->max_split_rows; r.maxc = cur->max_split_cols;
      r.kind_prev = l > 0 ? (cur - 1)->kind : cur->kind;
    }
    __syncthreads();
    const RecBuf& rec = sm.rec;
    // ---- 1. Q[x][m] for every subset m of the levels ------------------------------------------------------------------
    for (int e = tid; e < 5 << D; e += kFoldNT) {
      const int x = e >> D, m = e & ((1 << D) - 1);
      int64_t f = 1;
      for (int d = 0; d < D; ++d)
        if (m >> d & 1) f *= mp.size[d];
      // (f <= 2^20; a power of two on the usual machines: an add and a shift instead of a 64-bit division)
      sm.Q[x][m] = (f & (f - 1)) == 0 ? (rec.X[x] + f - 1) >> (63 - __clzll(f)) : (rec.X[x] + f - 1) / f;
    }
    __syncthreads();
    // ---- 2. VP[j] = weight-gradient all-reduce + penalty ------------------------------------------------
    for (int j = tid; j < K; j += kFoldNT) {
      uint32_t sI, sW, sO;
      const bool valid = fold_states(rec.kind, sm.dig[j], D, sI, sW, sO);
      int64_t v = 0, mem = 0, rs = 1, cs = 1;
      if (valid) {
        uint32_t w0 = 0, w1 = 0, i0 = 0, i1 = 0, o0 = 0, o1 = 0;
        for (int d = 0; d < D; ++d) {
          const int w = sW >> (2 * d) & 3, i = sI >> (2 * d) & 3, o = sO >> (2 * d) & 3;
          if (w == kS0) w0 |= 1u << d;
          if (w == kS1) w1 |= 1u << d;
          if (i == kS0) i0 |= 1u << d;
          if (i == kS1) i1 |= 1u << d;
          if (o == kS0) o0 |= 1u << d;
          if (o == kS1) o1 |= 1u << d;
          if (i == kS0 || o == kS0) rs *= mp.size[d];
          if (o == kS1) cs *= mp.size[d];
        }
        if (rec.kind == AUTODDL_GEMM) {
          const int64_t nw = sm.Q[1][w0] * sm.Q[2][w1];
          for (int d = 0; d < D; ++d)
            if ((sW >> (2 * d) & 3) == kB) {
              const int64_t p = mp.size[d], n = nw * (int64_t)rec.wgb;
              if (p > 1) v += (2 * p - 1) * mp.alpha[d] + 2 * (p - 1) * cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d];
            }
          mem = nw * (int64_t)rec.wsb;
        }
        mem += (sm.Q[3][i0] * sm.Q[4][i1] + sm.Q[0][o0] * sm.Q[2][o1]) * (int64_t)rec.eb;
      }
      const bool ok = valid && rs <= rec.maxr && cs <= rec.maxc && (mp.mem_cap == 0 || mem <= cap_layer);
      sm.VP[j] = v + (ok ? 0 : AUTODDL_PEN);
      if (node && chunk == 0) node[(size_t)tile * K + j] = v;
      if (mask && chunk == 0) mask[(size_t)tile * K + j] = ok ? 1 : 0;
    }
    __syncthreads();
    // ---- 3. the cells: forward + backward redistribution (R5), once per micro-batch (R25) -------------------------------------
    int64_t* out = T + (size_t)tile * K * K;
    const int per = (K * K + chunks - 1) / chunks, c_end = (chunk + 1) * per < K * K ? (chunk + 1) * per : K * K;
    for (int c = chunk * per + tid; c < c_end; c += kFoldNT) {
      const int i = c / K, j = c % K;
      int64_t e = 0;
      if (l > 0) {
        if (sm.ok[rec.kind_prev][i] && sm.ok[rec.kind][j])
          e = fold_walk(sm.stO[rec.kind_prev][i], sm.stI[rec.kind][j], sm.Q[3], sm.Q[4], rec.eb, sm) +
              fold_walk(sm.duI[rec.kind][j], sm.duO[rec.kind_prev][i], sm.Q[3], sm.Q[4], rec.eb, sm);
      }
      out[c] = mp.accum * e + sm.VP[j];
    }
  }
}

}  // namespace

int launch_build_tables_folded(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int64_t* d_T,
                               int64_t* d_node, uint8_t* d_mask, cudaStream_t st) {
  const int64_t nt = (int64_t)Bp * L;
  if (nt > 0x7fffffff) { set_error("Bp*L too large"); return AUTODDL_EINVAL; }
  const int slots = device_sm_count() * 4;
  int chunks = (int)((2 * slots + nt - 1) / nt);                         // few tiles: split them into blocks of cells
  const int max_chunks = (mp.K * mp.K + kFoldNT - 1) / kFoldNT;          // (at least one cell per thread)
  if (chunks > max_chunks) chunks = max_chunks;
  if (chunks < 1) chunks = 1;
  if (nt * chunks > 0x7fffffff) chunks = 1;
  const int64_t units = nt * chunks;
  const int grid = (int)(units < slots ? units : slots);
  build_tables_folded_kernel<<<grid, kFoldNT, 0, st>>>(d_layers, (int)nt, L, chunks, mp, d_T, d_node, d_mask);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
