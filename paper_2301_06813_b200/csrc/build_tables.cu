// (a1) SBP cost-table builder for sm_100a.
//
// T[p][l][i][j] = E(l,i,j) + V(l,j) + PEN*[j infeasible at l]      (R8)
//   E: forward + backward redistribution of layer l's input between producer-output signature i
//      and consumer-input signature j (collectives Table 2, PAPER.md:102-108;
//      link class per mesh level)
//   V: all-reduce of the weight gradient on every level where W is replicated
//   feasibility: split limits and per-device memory
//
// Design (differs from a per-cell evaluation on purpose).  A redistribution moves
// every mesh level through a fixed sequence of states -- after the free slice, after reduce-scatter,
// after all-to-all, after all-gather -- that depends only on the level's own (from, to) pair; levels
// interact only through the local tensor size at the moment a collective runs.  Per K x K tile:
//   1. Q[x][m] = ceil(x / prod(levels in m)) for the five extents and every level subset (magic-number
//      division: divisors are fixed per launch)
//   2. per level d and split configuration cfg (3^D of them): gather/scatter cost CG, all-to-all cost CA
//      of the input tensor, all-reduce cost of the weight gradient, local sizes of W and O
//   3. R[a][b] over the 4^D x 4^D state vectors = a sum of <= 3D table entries whose addresses do not
//      depend on the tile (hoisted out of the persistent tile loop when one thread owns one entry);
//      VP[j] = node cost + penalty per consumer signature from the step-2 tables
//   4. Esym[a][b] = R[a][b] + R[dual b][dual a]   (forward leg + backward leg)
//   5. the K x K expansion T[i][j] = Esym[O-state(i)][I-state(j)] + VP[j]: one shared-memory gather and one
//      64-bit add per cell, 16-byte streaming stores; all indices are hoisted out of the tile loop.
// The kernel is then bound by the HBM write of 8 B per cell instead of integer arithmetic.
#include "sbp_builder.cuh"

namespace autoddl {

namespace {

// ======================================================================================================
// Generic kernel (any D; used for D = 1 and D = 3): one tile per loop iteration, direct 16-byte stores.
// ======================================================================================================
template <int D>
struct TileSmem {
  static constexpr int K = Pow<D>::K, NS = Pow<D>::NS, NC = Pow<D>::NC;
  int64_t Q[5][8];                                      // M, Kd, N, in_rows, in_cols  x  level subset
  int64_t CG[D][NC + 1];                                // [..][NC] = 0: the slot that does not run
  int64_t CA[D][NC + 1];
  int64_t WAR[D][NC];
  int64_t locW[NC], locO[NC];
  alignas(16) int64_t VP[K];
  alignas(16) int64_t E[NS * NS];
  RecBuf rec[2];
  SigInfo sig[2][K];
};

template <int D>
__global__ void __launch_bounds__(256)
build_tables_kernel(const autoddl_layer* __restrict__ layers, int ntiles, int L, MeshParams mp,
                    int64_t* __restrict__ T, int64_t* __restrict__ node, uint8_t* __restrict__ mask) {
  using SM = TileSmem<D>;
  constexpr int K = Pow<D>::K, NS = Pow<D>::NS, NC = Pow<D>::NC, NT = 256, KH = K / 2;
  static_assert(D * NC <= 96 && 192 + NC <= NT && (5 << D) <= NT, "role layout");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);
  const int tid = threadIdx.x;

  fill_sig_table<D>(sm.sig, mp, tid, NT);
  if (tid < D) { sm.CG[tid][NC] = 0; sm.CA[tid][NC] = 0; }
  __syncthreads();

  // step 1 role: (extent, level subset); step 2 roles: A [0,96) B [96,192) C [192,..)
  const int q_x = tid >> D, q_m = tid & ((1 << D) - 1);
  const int role_base = tid < 96 ? 0 : (tid < 192 ? 96 : 192);
  const int role_i = tid - role_base;
  const int role_d = role_i / NC, role_cfg = role_i % NC;
  int role_m0 = 0, role_m1 = 0;
  cfg_masks<D>(role_cfg, role_m0, role_m1);
  const int64_t cap_layer = mp.mem_cap / L;

  int tile = blockIdx.x;
  if (tile >= ntiles) return;
  auto stage = [&](int b, int tl) {                         // thread `part` stages 16-byte part (or the previous kind)
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

    // ---- 1. Q[x][m]: x = M, Kd, N, in_rows, in_cols (the record's first five int64) ---------------------
    if (tid < (5 << D)) sm.Q[q_x][q_m] = cdiv_magic(rec.X[q_x], (uint32_t)mp.sub[q_m], mp.magic_sub[q_m]);
    __syncthreads();

    // ---- 2. tables per level and split configuration -------------------------------------------------------
    if (role_base == 0 && role_i < D * NC) {
      if (l > 0) {                                           // input tensor: Table 2 rows 2 and 3
        const int d = role_d;
        const int64_t n = sm.Q[3][role_m0] * sm.Q[4][role_m1] * (int64_t)rec.eb;
        const int64_t p = mp.size[d];
        int64_t cg = 0, ca = 0;
        if (p > 1) {
          cg = mp.accum * ((p - 1) * (mp.alpha[d] + cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d]));
          ca = mp.accum * ((p - 1) * mp.alpha[d] + n * mp.beta[d]);      // R25: once per micro-batch
        }
        sm.CG[d][role_cfg] = cg;
        sm.CA[d][role_cfg] = ca;
      }
    } else if (role_base == 96 && role_i < D * NC) {
      if (rec.kind == AUTODDL_GEMM) {                        // weight gradient: AllReduce row
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

    // ---- 3. VP[j] (node cost + penalty) and R[a][b] ------------------------------------------------------------
    for (int j = tid; j < K; j += NT) {
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
      sm.VP[j] = v + (ok ? 0 : AUTODDL_PEN);
      const size_t o = (size_t)tile * K + j;
      if (node) node[o] = v;
      if (mask) mask[o] = ok ? 1 : 0;
    }
    if (l > 0) {
      const int64_t* tab = &sm.CG[0][0];
      for (int e = tid; e < NS * NS; e += NT) {
        int idx[3 * D];
        r_slots<D>(e / NS, e % NS, idx);
        int64_t c = 0;
#pragma unroll
        for (int k = 0; k < 3 * D; ++k) c += tab[idx[k]];
        sm.E[e] = c;
      }
    }
    __syncthreads();

    // ---- 4. K x K expansion: forward leg R[a][b] + backward leg R[dual b][dual a] + VP[j] ---------------------
    int64_t* out = T + (size_t)tile * K * K;
    for (int c = tid; c < K * KH; c += NT) {
      const int i = c / KH, j = (c % KH) * 2;
      longlong2 v = make_longlong2(sm.VP[j], sm.VP[j + 1]);
      if (l > 0) {
        const int a = sm.sig[rec.kind_prev][i].a_idx;
        if (a < NS) {
          const int da = dual_vec<D>(a);
          const SigInfo& s0 = sm.sig[rec.kind][j];
          const SigInfo& s1 = sm.sig[rec.kind][j + 1];
          if (s0.b_idx >= 0) v.x += sm.E[a * NS + s0.b_idx] + sm.E[s0.db_idx * NS + da];
          if (s1.b_idx >= 0) v.y += sm.E[a * NS + s1.b_idx] + sm.E[s1.db_idx * NS + da];
        }
      }
      __stcs(reinterpret_cast<longlong2*>(out + (size_t)i * K + j), v);
    }
    if (tid < 5) cp_async_wait_all();
    __syncthreads();                                       // E is rewritten by the next tile's step 3; publishes the record
  }
}

// ======================================================================================================
// Four and five mesh levels (R26; 2 nodes x 16 GPUs = 2 | 2.2.2.2): K <= 256 signatures over
// the allowed rows only.  The 4^D x 4^D state table of the kernels above no longer fits shared memory (8 MB at D = 5),
// so every cell sums its <= 6D table entries itself:  T[i][j] = VP[j] + R[a(i)][b(j)] + R[dual b(j)][dual a(i)],
// R = sum of the reduce-scatter / all-to-all / all-gather entries of steps 1-2 that the levels' walks select.
// A work unit is a block of rows of one tile (a tile is split so that a single chain still fills the machine).
// ======================================================================================================
template <int D>
struct DirectSmem {
  static constexpr int NC = Pow<D>::NC;
  int64_t Q[5][1 << D];
  int64_t CG[D][NC + 1];                                // [..][NC] = 0: the slot that does not run
  int64_t CA[D][NC + 1];
  int64_t WAR[D][NC];
  int64_t locW[NC], locO[NC];
  int64_t VP[256];
  RecBuf rec;
  uint32_t walk[16];
  SigInfo sig[2][256];
};

// facts per (layer kind, signature) with the mixed-radix index over the allowed rows
template <int D>
__device__ __forceinline__ void fill_sig_table_compact(SigInfo (*sig)[256], const MeshParams& mp, int K, int tid, int nthreads) {
  constexpr int NS = Pow<D>::NS;
  for (int x = tid; x < 2 * K; x += nthreads) {
    const int kind = x / K, j = x % K;
    int dig[D], r = j;
#pragma unroll
    for (int d = D - 1; d >= 0; --d) {                     // level 0 most significant; digit = rank among the allowed rows
      const int nr = __popc(mp.allow[d]);
      int xr = r % nr;
      r /= nr;
      int g = 0;
      for (int t = 0; t < 6; ++t)
        if ((mp.allow[d] >> t) & 1) {
          if (xr == 0) { g = t; break; }
          --xr;
        }
      dig[d] = g;
    }
    SigInfo si{};
    int a = 0, b = 0, cw = 0, co = 0, pw = 1, rs = 1, cs = 1;
    bool valid = true;
#pragma unroll
    for (int d = 0; d < D; ++d) {
      const int g = dig[d];
      int sI, sO, sW;
      if (kind == AUTODDL_GEMM) { sI = c_gemm_I[g]; sO = c_gemm_O[g]; sW = c_gemm_W[g]; }
      else { sI = sO = c_attn_IO[g]; sW = kB; if (sI < 0) { valid = false; sI = sO = kB; } }
      a = a * 4 + sO;
      b = b * 4 + sI;
      cw += (sW == kS0 ? 1 : sW == kS1 ? 2 : 0) * pw;
      co += (sO == kS0 ? 1 : sO == kS1 ? 2 : 0) * pw;
      pw *= 3;
      if (sI == kS0) si.mI0 |= 1 << d;
      if (sI == kS1) si.mI1 |= 1 << d;
      if (sW == kB) si.wB |= 1 << d;
      if (sI == kS0 || sO == kS0) rs *= mp.size[d];
      if (sO == kS1) cs *= mp.size[d];
    }
    si.a_idx = valid ? a : NS;
    si.b_idx = valid ? b : -1;
    si.db_idx = valid ? dual_vec<D>(b) : -1;
    si.cfgW = cw; si.cfgO = co; si.valid = valid; si.allowed = 1; si.rowsplit = rs; si.colsplit = cs;
    sig[kind][j] = si;
  }
}

constexpr int kDirectNT = 512;

template <int D>
__global__ void __launch_bounds__(kDirectNT)
build_tables_direct_kernel(const autoddl_layer* __restrict__ layers, int ntiles, int L, int K, int chunks, MeshParams mp,
                           int64_t* __restrict__ T, int64_t* __restrict__ node, uint8_t* __restrict__ mask) {
  using SM = DirectSmem<D>;
  constexpr int NS = Pow<D>::NS, NC = Pow<D>::NC, NT = kDirectNT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);
  const int tid = threadIdx.x;

  fill_sig_table_compact<D>(sm.sig, mp, K, tid, NT);
  if (tid < D) { sm.CG[tid][NC] = 0; sm.CA[tid][NC] = 0; }
  if (tid < 16) sm.walk[tid] = c_walk.w[tid];
  const int64_t cap_layer = mp.mem_cap / L;
  const int rows_per_chunk = (K + chunks - 1) / chunks;
  int last_tile = -1;

  for (int unit = blockIdx.x; unit < ntiles * chunks; unit += gridDim.x) {
    const int tile = unit / chunks, chunk = unit % chunks;
    const int l = tile % L;
    __syncthreads();                                         // previous unit's readers are done with the tables
    if (tile != last_tile) {
      last_tile = tile;
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
      // ---- 1. Q[x][m] ----------------------------------------------------------------------------------------
      if (tid < (5 << D)) {
        const int x = tid >> D, m = tid & ((1 << D) - 1);
        sm.Q[x][m] = cdiv_magic(rec.X[x], (uint32_t)mp.sub[m], mp.magic_sub[m]);
      }
      __syncthreads();
      // ---- 2. tables per level and split configuration (Table 2) ------------------------------
      for (int e = tid; e < D * NC; e += NT) {
        const int d = e / NC, cfg = e % NC;
        int m0, m1;
        cfg_masks<D>(cfg, m0, m1);
        const int64_t p = mp.size[d];
        int64_t cg = 0, ca = 0, war = 0;
        if (p > 1) {
          const int64_t n = sm.Q[3][m0] * sm.Q[4][m1] * (int64_t)rec.eb;
          cg = mp.accum * ((p - 1) * (mp.alpha[d] + cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d]));
          ca = mp.accum * ((p - 1) * mp.alpha[d] + n * mp.beta[d]);      // R25: once per micro-batch
          const int64_t nw = sm.Q[1][m0] * sm.Q[2][m1] * (int64_t)rec.wgb;
          war = (2 * p - 1) * mp.alpha[d] + 2 * (p - 1) * cdiv_magic(nw, (uint32_t)p, mp.magic_size[d]) * mp.beta[d];
        }
        sm.CG[d][cfg] = cg;
        sm.CA[d][cfg] = ca;
        sm.WAR[d][cfg] = war;
        if (d == 0) {
          sm.locW[cfg] = sm.Q[1][m0] * sm.Q[2][m1];
          sm.locO[cfg] = sm.Q[0][m0] * sm.Q[2][m1];
        }
      }
      __syncthreads();
      // ---- 3. VP[j] = node cost + penalty ----------------------------------------------------------------------
      for (int j = tid; j < K; j += NT) {
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
        const bool ok = si.valid && si.rowsplit <= rec.maxr && si.colsplit <= rec.maxc && (mp.mem_cap == 0 || mem <= cap_layer);
        sm.VP[j] = v + (ok ? 0 : AUTODDL_PEN);
        if (chunk == 0) {                                      // one unit per tile reports the node costs and the mask
          const size_t o = (size_t)tile * K + j;
          if (node) node[o] = v;
          if (mask) mask[o] = ok ? 1 : 0;
        }
      }
      __syncthreads();
    }
    // ---- 4. the cells of this unit's rows ------------------------------------------------------------------------
    const RecBuf& rec = sm.rec;
    const int r0 = chunk * rows_per_chunk;
    const int r1 = r0 + rows_per_chunk < K ? r0 + rows_per_chunk : K;
    const int64_t* tab = &sm.CG[0][0];
    int64_t* out = T + (size_t)tile * K * K;
    for (int i = r0 + (tid >> 5); i < r1; i += NT / 32) {   // one warp per row: no division, the row's state vector once
      const int a = l > 0 ? sm.sig[rec.kind_prev][i].a_idx : NS;
      const int da = dual_vec<D>(a & (NS - 1));
      for (int j = tid & 31; j < K; j += 32) {
        int64_t v = sm.VP[j];
        const SigInfo& sj = sm.sig[rec.kind][j];
        if (a < NS && sj.b_idx >= 0) {
          int idx[3 * D];
          r_slots<D>(a, sj.b_idx, idx, sm.walk);             // forward leg
#pragma unroll
          for (int k = 0; k < 3 * D; ++k) v += tab[idx[k]];
          r_slots<D>(sj.db_idx, da, idx, sm.walk);           // backward leg
#pragma unroll
          for (int k = 0; k < 3 * D; ++k) v += tab[idx[k]];
        }
        __stcs(out + (size_t)i * K + j, v);
      }
    }
  }
}

// ======================================================================================================
// K = 36 kernel (two mesh levels): distinct rows in shared memory, TMA bulk stores to global.
//
// A tile has only 16 distinct rows: row i depends on i through the producer's output state vector a(i),
// and the per-level output states of signatures 2, 4, 5 coincide (all P; for ATTN all invalid).  With
// class(i0) = {0,1,2,3,2,2}[i0] over the level-0 digit, rows 6*i0 .. 6*i0+5 of the tile equal the block
// EV[class(i0)][0..5][.] of 6 x 36 cells.  Per tile the CTA computes the 24 x 36 block rows
//   EV[r][j] = VP[j] + R[a(r)][b(j)] + R[dual b(j)][dual a(r)]
// in shared memory and one thread issues six 1,728-byte cp.async.bulk shared->global copies (SASS UBLKCP);
// the store stream runs on the TMA engine while the CTA prepares the next group of tiles (EV is double
// buffered; cp.async.bulk.wait_group.read guards its reuse).  G = 4 tiles share one barrier sequence.
// ======================================================================================================
template <int G_>
struct Smem36 {
  static constexpr int D = 2, K = 36, NS = 16, NC = 9, G = G_, ES = NS + 1, NROW = 24, STRIDE = NC + 1;
  struct PerTile {
    int64_t Q[5][4];                                    // M, Kd, N, in_rows, in_cols  x  level subset
    int64_t TAB[2 * D * STRIDE];                        // CG[D][NC+1] then CA[D][NC+1]; [..][NC] = 0
    int64_t WAR[D][NC];
    int64_t locW[NC], locO[NC];
    alignas(16) int64_t VP[K];
    alignas(16) int64_t E[ES * ES];                     // R[a][b]; row NS and column NS stay 0
  };
  alignas(128) int64_t EV[2][G][NROW * K];
  PerTile t[G];
  RecBuf rec[2][G];
  SigInfo sig[2][K];
  int32_t meta[2];                                      // (kind | kind_prev << 1) of the group's tiles, 2 bits each
};

__device__ __forceinline__ void bulk_s2g(void* dst_gmem, const void* src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes)
               : "memory");
}

// Work of one team (CTA): groups blockIdx.x, blockIdx.x + gridDim.x, ... of up to G consecutive tiles of the flat tile
// list (a group may straddle chains)
struct GroupSched {
  int tile0, l0, nt;         // first tile, its layer index, tiles in the group
  bool valid;
  int ntiles, L, step, l_step;
  __device__ __forceinline__ void init(int ntiles_, int L_, int G) {
    ntiles = ntiles_; L = L_; step = gridDim.x;
    tile0 = blockIdx.x * G; valid = tile0 < ntiles;
    l0 = (int)(((int64_t)blockIdx.x * G) % L);
    l_step = (int)(((int64_t)gridDim.x * G) % L);
    nt = ntiles - tile0 < G ? ntiles - tile0 : G;
  }
  __device__ __forceinline__ void advance(int G) {
    tile0 += step * G;
    valid = tile0 < ntiles;
    l0 += l_step;
    if (l0 >= L) l0 -= L;
    nt = ntiles - tile0 < G ? ntiles - tile0 : G;
  }
};

// NT builder threads, G tiles per group.
template <int NT, int G>
__global__ void __launch_bounds__(NT, 768 / NT)
build_tables36_kernel(const autoddl_layer* __restrict__ layers, int ntiles, int L, MeshParams mp,
                      int64_t* __restrict__ T, int64_t* __restrict__ node, uint8_t* __restrict__ mask) {
  using SM = Smem36<G>;
  constexpr int D = 2, K = SM::K, NS = SM::NS, NC = SM::NC, ES = SM::ES, NROW = SM::NROW;
  constexpr int STRIDE = SM::STRIDE;
  constexpr int NR = NS * NS / NT;                         // R entries per thread
  constexpr int RS = NT / K, EVN = (NROW + RS - 1) / RS;   // EV: row stride between a thread's rows, rows per thread
  constexpr int ISSUER = NT - 1;                           // idle in step 4 (RS * K < NT threads fill EV)
  constexpr int RA = G * D * NC;                           // threads of step-2 roles A and B; role C has G * NC
  static_assert(NS * NS % NT == 0 && RS * K < NT, "thread layout");
  static_assert(2 * RA + G * NC <= NT && G * 5 * (1 << D) <= NT && G * K <= NT && 5 * G <= NT, "role layout");
  extern __shared__ __align__(128) unsigned char smem36_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem36_raw);
  const int tid = threadIdx.x;

  {
    fill_sig_table<D>(sm.sig, mp, tid, NT);
    for (int x = tid; x < G * ES * ES; x += NT) sm.t[x / (ES * ES)].E[x % (ES * ES)] = 0;
    for (int x = tid; x < G * 2 * D; x += NT) sm.t[x / (2 * D)].TAB[(x % (2 * D)) * STRIDE + NC] = 0;
  }
  __syncthreads();
  auto bsync = [&]() { __syncthreads(); };

  GroupSched sc;
  sc.init(ntiles, L, G);

  // ---- tile-invariant roles of this thread ---------------------------------------------------------------
  // step 3: thread sums the <= 6 table entries of R[a][b] for NR state pairs (a, b) = tid + k * NT
  int slot[NR][3 * D];
  int e_own[NR];
#pragma unroll
  for (int k = 0; k < NR; ++k) {
    const int e = tid + k * NT;
    r_slots<D>(e / NS, e % NS, slot[k]);
    e_own[k] = (e / NS) * ES + e % NS;
  }
  // step 4: thread (r0, j) fills EV rows r0, r0 + RS, ... of column j; indices for GEMM -> GEMM edges
  const int ev_j = tid % K, ev_r0 = tid / K;               // ev_r0 >= RS: no rows
  int ev_idx[EVN];
  {
    const int b = sm.sig[0][ev_j].b_idx, db = sm.sig[0][ev_j].db_idx;
#pragma unroll
    for (int k = 0; k < EVN; ++k) {
      const int r = ev_r0 + RS * k;
      const int a = sm.sig[0][r < NROW ? r : 0].a_idx;      // block row r = class representative i0 = r / 6, i1 = r % 6
      ev_idx[k] = (a * ES + b) | (db * ES + dual_vec<D>(a)) << 16;
    }
  }
  // step 1 role: (tile in group, extent, level subset); step 2 roles: A [0,RA) B [RA,2RA) C [2RA,..)
  const int q_t = tid / (5 << D), q_x = (tid % (5 << D)) >> D, q_m = tid & ((1 << D) - 1);
  const int role_base = tid < RA ? 0 : (tid < 2 * RA ? RA : 2 * RA);
  const int role_i = tid - role_base;
  const int role_t = role_base == 2 * RA ? role_i / NC : role_i / (D * NC);   // tile in group
  const int role_d = (role_i % (D * NC)) / NC;                                // level (roles A, B)
  const int role_cfg = role_i % NC;
  int role_m0 = 0, role_m1 = 0;
  cfg_masks<D>(role_cfg, role_m0, role_m1);
  const int vp_t = tid / K, vp_j = tid % K;                // step 3: VP role (tid < G * K)
  const int64_t cap_layer = mp.mem_cap / L;

  if (!sc.valid) return;
  int buf = 0;
  // records: thread 5*t + part stages 16-byte part (or the previous kind) of tile t of the group
  auto stage_group = [&](int b, int tile_first, int lfirst) {
    if (tid < 5 * G) {
      const int t = tid / 5, part = tid % 5;
      int tile = tile_first + t;
      if (tile >= ntiles) tile = ntiles - 1;                // ragged tail: restage a valid record, never used
      int l = lfirst + t;
      while (l >= L) l -= L;
      const autoddl_layer* cur = layers + tile;
      RecBuf* dst = &sm.rec[b][t];
      if (part < 4) cp_async16(reinterpret_cast<unsigned char*>(dst) + 16 * part, reinterpret_cast<const unsigned char*>(cur) + 16 * part);
      else cp_async4(&dst->kind_prev, &(l > 0 ? cur - 1 : cur)->kind);
    }
  };
  auto pack_meta = [&](int b) {                             // after the records of buffer b have landed and are published
    int m = 0;
#pragma unroll
    for (int t = 0; t < G; ++t) m |= (sm.rec[b][t].kind | sm.rec[b][t].kind_prev << 1) << (2 * t);
    sm.meta[b] = m;
  };
  stage_group(0, sc.tile0, sc.l0);
  cp_async_wait_all();
  bsync();
  if (tid == 0) pack_meta(0);

  for (int it = 0; sc.valid; ++it) {
    const int tile0 = sc.tile0, nt = sc.nt, l0 = sc.l0;
    sc.advance(G);                                            // sc now describes the next group
    stage_group(buf ^ 1, sc.valid ? sc.tile0 : tile0, sc.valid ? sc.l0 : l0);
    int first = 0;                                            // bit t: tile t of the group is a chain's layer 0
    {
      int l = l0;
#pragma unroll
      for (int t = 0; t < G; ++t) {
        first |= (l == 0) << t;
        l = (l + 1 == L) ? 0 : l + 1;
      }
    }
    const int eb = it & 1;

    // ---- 1. Q[x][m]: x = M, Kd, N, in_rows, in_cols (the record's first five int64) ---------------------
    if (tid < G * (5 << D) && q_t < nt)
      sm.t[q_t].Q[q_x][q_m] = cdiv_magic(sm.rec[buf][q_t].X[q_x], (uint32_t)mp.sub[q_m], mp.magic_sub[q_m]);
    bsync();

    // ---- 2. tables per level and split configuration -------------------------------------------------------
    if (role_t < nt) {
      typename SM::PerTile& pt = sm.t[role_t];
      const RecBuf& rec = sm.rec[buf][role_t];
      if (role_base == 0) {
        if (!(first >> role_t & 1)) {                        // input tensor: Table 2 rows 2 and 3
          const int d = role_d;
          const int64_t n = pt.Q[3][role_m0] * pt.Q[4][role_m1] * (int64_t)rec.eb;
          const int64_t p = mp.size[d];
          int64_t cg = 0, ca = 0;
          if (p > 1) {
            cg = mp.accum * ((p - 1) * (mp.alpha[d] + cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d]));
            ca = mp.accum * ((p - 1) * mp.alpha[d] + n * mp.beta[d]);      // R25: once per micro-batch
          }
          pt.TAB[d * STRIDE + role_cfg] = cg;
          pt.TAB[(D + d) * STRIDE + role_cfg] = ca;
        }
      } else if (role_base == RA) {
        if (rec.kind == AUTODDL_GEMM) {                      // weight gradient: AllReduce row
          const int d = role_d;
          const int64_t n = pt.Q[1][role_m0] * pt.Q[2][role_m1] * (int64_t)rec.wgb;
          const int64_t p = mp.size[d];
          pt.WAR[d][role_cfg] =
              p > 1 ? (2 * p - 1) * mp.alpha[d] + 2 * (p - 1) * cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d] : 0;
        }
      } else if (role_i < G * NC) {
        pt.locW[role_cfg] = pt.Q[1][role_m0] * pt.Q[2][role_m1];
        pt.locO[role_cfg] = pt.Q[0][role_m0] * pt.Q[2][role_m1];
      }
    }
    bsync();

    // ---- 3. VP[j] (node cost + penalty) and R[a][b] (zero for a chain's first layer: no producer) -----------------
    if (tid < G * K && vp_t < nt) {
      typename SM::PerTile& pt = sm.t[vp_t];
      const RecBuf& rec = sm.rec[buf][vp_t];
      const SigInfo si = sm.sig[rec.kind][vp_j];
      int64_t v = 0, mem = 0;
      if (si.valid) {
        if (rec.kind == AUTODDL_GEMM) {
#pragma unroll
          for (int d = 0; d < D; ++d)
            if (si.wB >> d & 1) v += pt.WAR[d][si.cfgW];
          mem = pt.locW[si.cfgW] * (int64_t)rec.wsb;
        }
        mem += (pt.Q[3][si.mI0] * pt.Q[4][si.mI1] + pt.locO[si.cfgO]) * (int64_t)rec.eb;
      }
      const bool ok = si.valid && si.allowed && si.rowsplit <= rec.maxr && si.colsplit <= rec.maxc && (mp.mem_cap == 0 || mem <= cap_layer);
      pt.VP[vp_j] = v + (ok ? 0 : AUTODDL_PEN);
      const size_t o = (size_t)(tile0 + vp_t) * K + vp_j;
      if (node) node[o] = v;
      if (mask) mask[o] = ok ? 1 : 0;
    }
#pragma unroll
    for (int t = 0; t < G; ++t) {
      if (t < nt) {
        const int64_t* tab = sm.t[t].TAB;
#pragma unroll
        for (int q = 0; q < NR; ++q) {
          int64_t c = 0;
          if (!(first >> t & 1)) {
#pragma unroll
            for (int k = 0; k < 3 * D; ++k) c += tab[slot[q][k]];
          }
          sm.t[t].E[e_own[q]] = c;
        }
      }
    }
    bsync();

    // ---- 4. EV[r][j] = VP[j] + R[a(r)][b(j)] + R[dual b(j)][dual a(r)]: the 24 block rows of every tile ---------------
    const int meta = sm.meta[buf];
    if (ev_r0 < RS) {
      if (meta == 0) {                                       // every edge of the group is GEMM -> GEMM: hoisted indices
#pragma unroll
        for (int t = 0; t < G; ++t) {
          if (t < nt) {
            const int64_t* E = sm.t[t].E;
            const int64_t vp = sm.t[t].VP[ev_j];
            int64_t* ev = &sm.EV[eb][t][ev_j];
#pragma unroll
            for (int k = 0; k < EVN; ++k)
              if (ev_r0 + RS * k < NROW) ev[(ev_r0 + RS * k) * K] = vp + E[ev_idx[k] & 0xffff] + E[ev_idx[k] >> 16];
          }
        }
      } else {
        for (int t = 0; t < nt; ++t) {
          const int kind = (meta >> (2 * t)) & 1, kind_prev = (meta >> (2 * t + 1)) & 1;
          const int64_t* E = sm.t[t].E;
          const int64_t vp = sm.t[t].VP[ev_j];
          int b = sm.sig[kind][ev_j].b_idx, db = sm.sig[kind][ev_j].db_idx;
          if (b < 0) b = db = NS;                            // invalid consumer signature: zero column
          for (int r = ev_r0; r < NROW; r += RS) {
            const int a = sm.sig[kind_prev][r].a_idx;        // class representative: i0 = r / 6 in 0..3
            const int da = a < NS ? dual_vec<D>(a) : NS;      // invalid producer signature: zero row
            sm.EV[eb][t][r * K + ev_j] = vp + E[a * ES + b] + E[db * ES + da];
          }
        }
      }
    }
    if (T) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // EV written by the generic proxy, read by TMA
    if (tid < 5 * G) cp_async_wait_all();                    // the next group's records have landed; the barrier publishes them
    bsync();

    // ---- 5. six 1,728-byte bulk stores per tile; the copies run while the CTA prepares the next group -----------------
    if (T && tid == ISSUER) {
      for (int t = 0; t < nt; ++t) {
        int64_t* out = T + (size_t)(tile0 + t) * K * K;
        const int64_t* src = sm.EV[eb][t];
#pragma unroll
        for (int i0 = 0; i0 < 6; ++i0) {
          const int cls = i0 < 4 ? i0 : 2;
          bulk_s2g(out + i0 * 6 * K, src + cls * 6 * K, 6 * K * 8);
        }
      }
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");   // the other EV buffer is free again
    }
    if (tid == 0) pack_meta(buf ^ 1);
    buf ^= 1;
  }
  if (T && tid == ISSUER) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// ======================================================================================================
// K = 216 kernel (three mesh levels): the same idea as the K = 36 kernel at one tile per iteration.
// A tile has 64 distinct rows (producer classes {0},{1},{3},{2,4,5} per level); the CTA fills EV[64][216] in shared
// memory (110 KB) and eight threads issue the 216 row copies of 1,728 bytes (cp.async.bulk shared -> global).  The
// 4096 x 9 slot indices of R[a][b] are decoded once per CTA into a byte table, so the per-tile R step is nine
// table reads per state pair.  The stores of a tile overlap steps 1-3 of the next one.
// ======================================================================================================
struct Smem216 {
  static constexpr int D = 3, K = 216, NS = 64, NC = 27, ES = NS + 1, NROW = 64, STRIDE = NC + 1;
  alignas(128) int64_t EV[NROW * K];
  alignas(16) int64_t E[ES * ES];                       // R[a][b]; row NS and column NS stay 0
  int64_t TAB[2 * D * STRIDE];                          // CG[D][NC+1] then CA[D][NC+1]; [..][NC] = 0
  int64_t Q[5][8];
  int64_t WAR[D][NC];
  int64_t locW[NC], locO[NC];
  alignas(16) int64_t VP[K];
  RecBuf rec[2];
  SigInfo sig[2][K];
  int16_t a_rc[2][NROW], da_rc[2][NROW];                // per producer kind: state vector of a row class, and its dual
  uint8_t slots[NS * NS][3 * D];                        // table entries whose sum is R[a][b]
};

__global__ void __launch_bounds__(256, 1)
build_tables216_kernel(const autoddl_layer* __restrict__ layers, int ntiles, int L, MeshParams mp,
                       int64_t* __restrict__ T, int64_t* __restrict__ node, uint8_t* __restrict__ mask) {
  using SM = Smem216;
  constexpr int D = 3, K = SM::K, NS = SM::NS, NC = SM::NC, ES = SM::ES, NROW = SM::NROW, STRIDE = SM::STRIDE, NT = 256;
  constexpr int NISS = 8, ISS0 = NT - 32;                  // issuing threads: the first 8 lanes of the last warp
  extern __shared__ __align__(128) unsigned char smem216_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem216_raw);
  const int tid = threadIdx.x;

  // ---- once per CTA --------------------------------------------------------------------------------------
  fill_sig_table<D>(sm.sig, mp, tid, NT);
  for (int x = tid; x < ES * ES; x += NT) sm.E[x] = 0;
  if (tid < 2 * D) sm.TAB[tid * STRIDE + NC] = 0;
  for (int e = tid; e < NS * NS; e += NT) {
    int idx[3 * D];
    r_slots<D>(e / NS, e % NS, idx);
#pragma unroll
    for (int k = 0; k < 3 * D; ++k) sm.slots[e][k] = (uint8_t)idx[k];
  }
  __syncthreads();
  if (tid < 2 * NROW) {                                    // row class rc = (c0, c1, c2), representative digits = classes
    const int kind = tid / NROW, rc = tid % NROW;
    const int i = (rc >> 4) * 36 + ((rc >> 2) & 3) * 6 + (rc & 3);
    const int a = sm.sig[kind][i].a_idx;
    sm.a_rc[kind][rc] = (int16_t)a;
    sm.da_rc[kind][rc] = (int16_t)(a < NS ? dual_vec<D>(a) : NS);
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

    // ---- 1. Q[x][m] -----------------------------------------------------------------------------------------
    if (tid < (5 << D)) sm.Q[q_x][q_m] = cdiv_magic(rec.X[q_x], (uint32_t)mp.sub[q_m], mp.magic_sub[q_m]);
    __syncthreads();

    // ---- 2. tables per level and split configuration -------------------------------------------------------
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

    // ---- 3. VP[j] and R[a][b] ---------------------------------------------------------------------------------
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
      sm.VP[j] = v + (ok ? 0 : AUTODDL_PEN);
      const size_t o = (size_t)tile * K + j;
      if (node) node[o] = v;
      if (mask) mask[o] = ok ? 1 : 0;
    }
    for (int e = tid; e < NS * NS; e += NT) {
      int64_t c = 0;
      if (l > 0) {
#pragma unroll
        for (int k = 0; k < 3 * D; ++k) c += sm.TAB[sm.slots[e][k]];
      }
      sm.E[(e / NS) * ES + e % NS] = c;
    }
    if (tid >= ISS0 && tid < ISS0 + NISS) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // EV is free again
    __syncthreads();

    // ---- 4. EV[rc][j] = VP[j] + R[a(rc)][b(j)] + R[dual b(j)][dual a(rc)] ------------------------------------------
    if (tid < K) {                                         // thread j fills column j of all 64 row classes
      const int j = tid, kind_prev = rec.kind_prev;
      int b = sm.sig[rec.kind][j].b_idx, db = sm.sig[rec.kind][j].db_idx;
      if (b < 0) b = db = NS;                              // invalid consumer signature: zero column
      const int64_t vp = sm.VP[j];
      const int64_t* Eb = sm.E + b;
      const int64_t* Ed = sm.E + db * ES;
#pragma unroll 8
      for (int rc = 0; rc < NROW; ++rc) {
        const int a = sm.a_rc[kind_prev][rc], da = sm.da_rc[kind_prev][rc];
        sm.EV[rc * K + j] = vp + Eb[a * ES] + Ed[da];
      }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (tid < 5) cp_async_wait_all();
    __syncthreads();

    // ---- 5. 216 row copies of 1,728 bytes, 27 per issuing thread ---------------------------------------------------
    if (tid >= ISS0 && tid < ISS0 + NISS) {
      int64_t* out = T + (size_t)tile * K * K;
      for (int i = tid - ISS0; i < K; i += NISS) {
        const int i0 = i / 36, i1 = (i / 6) % 6, i2 = i % 6;
        const int rc = (i0 < 4 ? i0 : 2) * 16 + (i1 < 4 ? i1 : 2) * 4 + (i2 < 4 ? i2 : 2);
        bulk_s2g(out + (size_t)i * K, sm.EV + rc * K, K * 8);
      }
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
  }
  if (tid >= ISS0 && tid < ISS0 + NISS) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

template <int D>
int launch_d(const autoddl_layer* d_layers, int ntiles, int L, const MeshParams& mp, int64_t* d_T,
             int64_t* d_node, uint8_t* d_mask, cudaStream_t st) {
  const size_t smem = sizeof(TileSmem<D>);
  if (smem > 48 * 1024)
    ADL_CUDA_CHECK(cudaFuncSetAttribute(build_tables_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int dev = 0, sms = 148;
  ADL_CUDA_CHECK(cudaGetDevice(&dev));
  ADL_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int per_sm = (D == 3) ? 1 : 4;
  const int grid = ntiles < sms * per_sm ? ntiles : sms * per_sm;     // persistent, grid-stride over tiles
  build_tables_kernel<D><<<grid, 256, smem, st>>>(d_layers, ntiles, L, mp, d_T, d_node, d_mask);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

int launch_216(const autoddl_layer* d_layers, int ntiles, int L, const MeshParams& mp, int64_t* d_T,
               int64_t* d_node, uint8_t* d_mask, cudaStream_t st) {
  const size_t smem = sizeof(Smem216);
  ADL_CUDA_CHECK(cudaFuncSetAttribute(build_tables216_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int dev = 0, sms = 148;
  ADL_CUDA_CHECK(cudaGetDevice(&dev));
  ADL_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int grid = ntiles < sms ? ntiles : sms;                        // persistent, one CTA per SM
  build_tables216_kernel<<<grid, 256, smem, st>>>(d_layers, ntiles, L, mp, d_T, d_node, d_mask);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

constexpr int kNT = 256, kG = 4;                  // tables only: 3 CTAs of 256 threads per SM, 4 tiles per group

int launch_36(const autoddl_layer* d_layers, int ntiles, int L, const MeshParams& mp, int64_t* d_T,
              int64_t* d_node, uint8_t* d_mask, cudaStream_t st) {
  auto kern = build_tables36_kernel<kNT, kG>;
  const size_t smem = sizeof(Smem36<kG>);
  ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int dev = 0, sms = 148;
  ADL_CUDA_CHECK(cudaGetDevice(&dev));
  ADL_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int ngroups = (ntiles + kG - 1) / kG;
  const int grid = ngroups < sms * 3 ? ngroups : sms * 3;             // persistent, grid-stride over tile groups
  kern<<<grid, kNT, smem, st>>>(d_layers, ntiles, L, mp, d_T, d_node, d_mask);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

template <int D>
int launch_direct(const autoddl_layer* d_layers, int ntiles, int L, const MeshParams& mp, int64_t* d_T,
                  int64_t* d_node, uint8_t* d_mask, cudaStream_t st) {
  auto kern = build_tables_direct_kernel<D>;
  const size_t smem = sizeof(DirectSmem<D>);
  if (smem > 48 * 1024) ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int dev = 0, sms = 148;
  ADL_CUDA_CHECK(cudaGetDevice(&dev));
  ADL_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int slots = sms * 2;                                           // two CTAs of 512 threads per SM
  int chunks = (2 * slots + ntiles - 1) / ntiles;                      // few tiles: split them into row blocks
  if (chunks > 8) chunks = 8;
  if (chunks > mp.K) chunks = mp.K;
  if (chunks < 1) chunks = 1;
  const int64_t units = (int64_t)ntiles * chunks;
  const int grid = (int)(units < slots ? units : slots);
  kern<<<grid, kDirectNT, smem, st>>>(d_layers, ntiles, L, mp.K, chunks, mp, d_T, d_node, d_mask);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace

int launch_build_tables(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int64_t* d_T,
                        int64_t* d_node, uint8_t* d_mask, cudaStream_t st) {
  const int64_t nt = (int64_t)Bp * L;
  if (nt > 0x7fffffff) { set_error("Bp*L too large"); return AUTODDL_EINVAL; }
  if (mp.fold) return launch_build_tables_folded(d_layers, Bp, L, mp, d_T, d_node, d_mask, st);
  switch (mp.ndim) {
    case 1: return launch_d<1>(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
    case 2: return launch_36(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
    case 3: {
      static const bool generic = ADL_DEBUG_ENV("AUTODDL_BT216_GENERIC");          // debug builds only
      if (generic) return launch_d<3>(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
      return launch_216(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
    }
    case 4: return launch_direct<4>(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
    case 5: return launch_direct<5>(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
  }
  set_error("ndim must be 1..5");
  return AUTODDL_EINVAL;
}

}  // namespace autoddl
