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
#include "common.cuh"

namespace autoddl {

namespace {

constexpr int kS0 = 0, kS1 = 1, kB = 2, kP = 3;

// per-level signature rows (PAPER.md:193 rows 0..2; replicate; partial pass-through), R1
__device__ __constant__ int8_t c_gemm_I[6] = {kS0, kB, kS1, kB, kP, kB};
__device__ __constant__ int8_t c_gemm_W[6] = {kB, kS1, kS0, kB, kB, kP};
__device__ __constant__ int8_t c_gemm_O[6] = {kS0, kS1, kP, kB, kP, kP};
__device__ __constant__ int8_t c_attn_IO[6] = {kS0, kS1, -1, kB, -1, -1};

// ---- one level's walk through a redistribution a -> b, packed ----------------------------------------
// bits 0-1 / 2-3 / 4-5 / 6-7: split code (0 none, 1 rows, 2 cols) after slice / reduce-scatter / all-to-all /
// all-gather; bit 8: reduce-scatter runs, bit 9: all-to-all runs, bit 10: all-gather runs.
constexpr bool cx_split(int s) { return s == kS0 || s == kS1; }
constexpr int cx_code(int s) { return s == kS0 ? 1 : (s == kS1 ? 2 : 0); }
constexpr uint32_t cx_walk(int a, int b) {
  const int s0 = (a == kB && cx_split(b)) ? b : a;                 // replicated -> split: keep own slice, free
  const bool r1 = (s0 == kP && b != kP);                           // partial -> anything else: reduce-scatter
  const int s1 = r1 ? (b == kB ? kS1 : b) : s0;
  const bool r2 = cx_split(s1) && cx_split(b) && s1 != b;          // change of split axis: all-to-all
  const int s2 = r2 ? b : s1;
  const bool r3 = cx_split(s2) && b == kB;                         // split -> replicated: all-gather
  const int s3 = r3 ? kB : s2;
  return (uint32_t)(cx_code(s0) | cx_code(s1) << 2 | cx_code(s2) << 4 | cx_code(s3) << 6 | (r1 ? 256 : 0) |
                    (r2 ? 512 : 0) | (r3 ? 1024 : 0));
}
struct WalkTable { uint32_t w[16]; };
constexpr WalkTable make_walks() {
  WalkTable t{};
  for (int a = 0; a < 4; ++a)
    for (int b = 0; b < 4; ++b) t.w[a * 4 + b] = cx_walk(a, b);
  return t;
}
__device__ __constant__ WalkTable c_walk = make_walks();

__device__ __forceinline__ int dual_of(int s) { return s == kB ? kP : (s == kP ? kB : s); }

// ceil(n / d) for n >= 0 with the launch-constant divisor d and M = ceil(2^64 / d): the multiply-high
// quotient is exact for n < 2^64 / d (d <= 2^20 is enforced by the API, so n < 2^43 is safe).
__device__ __forceinline__ int64_t cdiv_magic(int64_t n, uint32_t d, uint64_t M) {
  if (d == 1) return n;
  if ((uint64_t)n < (1ull << 43)) {
    const uint64_t q = __umul64hi((uint64_t)n, M);
    return (int64_t)(q + (q * d != (uint64_t)n));
  }
  return (n + d - 1) / d;
}

template <int D> struct Pow { };
template <> struct Pow<1> { static constexpr int K = 6, NS = 4, NC = 3; };
template <> struct Pow<2> { static constexpr int K = 36, NS = 16, NC = 9; };
template <> struct Pow<3> { static constexpr int K = 216, NS = 64, NC = 27; };

// Layer records are staged one tile ahead with cp.async into a double buffer in shared memory (80 bytes:
// the 64-byte record, then the previous layer's kind), so the tile loop never waits on a global load and
// no register is held across an iteration for the prefetch.
struct alignas(16) RecBuf {
  int64_t X[5];              // M, Kd, N, in_rows, in_cols
  int32_t kind, eb, wgb, wsb, maxr, maxc;
  int32_t kind_prev;
  int32_t pad[3];
};
static_assert(sizeof(RecBuf) == 80, "RecBuf mirrors autoddl_layer + 16 bytes");

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* dst_smem, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// per (layer kind, signature) facts, built once per CTA
struct SigInfo {
  int16_t a_idx;      // O state-vector index, or NS (zero-edge row) when the signature is invalid for the kind
  int16_t b_idx;      // I state-vector index, or -1
  int16_t db_idx;     // index of the dual of the I state vector (B <-> P), or -1
  uint8_t cfgW, cfgO; // split configuration of W / of O
  uint8_t mI0, mI1;   // level subsets splitting the input's rows / cols
  uint8_t wB;         // levels on which W is replicated
  uint8_t valid;
  int32_t rowsplit, colsplit;
};

template <int D>
struct TileSmem {
  static constexpr int K = Pow<D>::K, NS = Pow<D>::NS, NC = Pow<D>::NC;
  static constexpr bool kRows = (D <= 2);               // one thread per state pair: hoisted fast path
  static constexpr int G = kRows ? 4 : 1;               // tiles processed together per loop iteration
  struct PerTile {
    int64_t Q[5][8];                                    // M, Kd, N, in_rows, in_cols  x  level subset
    int64_t CG[D][NC + 1];                              // [..][NC] = 0: the slot that does not run
    int64_t CA[D][NC + 1];
    int64_t WAR[D][NC];
    int64_t locW[NC], locO[NC];
    alignas(16) int64_t VP[K];
    alignas(16) int64_t E[NS * NS];
    alignas(16) int64_t Esym[kRows ? (NS + 1) * (NS + 1) : 1];   // R[a][b] + R[dual b][dual a]; row NS, column NS = 0
  };
  RecBuf rec[2][G];
  SigInfo sig[2][K];
  alignas(16) PerTile t[G];
};


// split configuration index -> level subsets (rows, cols)
template <int D>
__device__ __forceinline__ void cfg_masks(int cfg, int& m0, int& m1) {
  m0 = m1 = 0;
#pragma unroll
  for (int e = 0; e < D; ++e) {
    const int sp = cfg % 3;
    cfg /= 3;
    if (sp == 1) m0 |= 1 << e;
    if (sp == 2) m1 |= 1 << e;
  }
}

// the <= 3D table entries whose sum is R[av][bv]; entries that do not run point at a zero slot
template <int D>
__device__ __forceinline__ void r_slots(int av, int bv, int (&idx)[3 * D]) {
  constexpr int NC = Pow<D>::NC, STRIDE = NC + 1, CA_OFF = D * STRIDE, ZERO = NC;
  int c0[D], c1[D], c2[D], c3[D];
  bool r1[D], r2[D], r3[D];
  int pw = 1;
#pragma unroll
  for (int d = 0; d < D; ++d) {
    const int sh = 2 * (D - 1 - d);
    const uint32_t w = c_walk.w[((av >> sh) & 3) * 4 + ((bv >> sh) & 3)];
    c0[d] = (w & 3) * pw; c1[d] = (w >> 2 & 3) * pw; c2[d] = (w >> 4 & 3) * pw; c3[d] = (w >> 6 & 3) * pw;
    r1[d] = w >> 8 & 1; r2[d] = w >> 9 & 1; r3[d] = w >> 10 & 1;
    pw *= 3;
  }
  int n = 0;
#pragma unroll
  for (int d = D - 1; d >= 0; --d) {        // reduce-scatter, innermost level first; message = tensor before it
    int cfg = 0;
#pragma unroll
    for (int e = 0; e < D; ++e) cfg += (e > d) ? c1[e] : (e < d ? c0[e] : 0);
    idx[n++] = r1[d] ? d * STRIDE + cfg : ZERO;
  }
#pragma unroll
  for (int d = D - 1; d >= 0; --d) {        // all-to-all, innermost first; message = tensor after it
    int cfg = 0;
#pragma unroll
    for (int e = 0; e < D; ++e) cfg += (e > d) ? c2[e] : (e < d ? c1[e] : c2[e]);
    idx[n++] = r2[d] ? CA_OFF + d * STRIDE + cfg : ZERO;
  }
#pragma unroll
  for (int d = 0; d < D; ++d) {             // all-gather, outermost first; message = tensor after it
    int cfg = 0;
#pragma unroll
    for (int e = 0; e < D; ++e) cfg += (e < d) ? c3[e] : (e > d ? c2[e] : 0);
    idx[n++] = r3[d] ? d * STRIDE + cfg : ZERO;
  }
}

template <int D>
__device__ __forceinline__ int dual_vec(int v) {
  int r = 0;
#pragma unroll
  for (int d = 0; d < D; ++d) r |= dual_of((v >> (2 * d)) & 3) << (2 * d);
  return r;
}

template <int D>
__global__ void __launch_bounds__(256, (D == 3) ? 1 : 3)
build_tables_kernel(const autoddl_layer* __restrict__ layers, int ntiles, int L, MeshParams mp,
                    int64_t* __restrict__ T, int64_t* __restrict__ node, uint8_t* __restrict__ mask) {
  using SM = TileSmem<D>;
  constexpr int K = Pow<D>::K, NS = Pow<D>::NS, NC = Pow<D>::NC, NT = 256, KH = K / 2, G = SM::G;
  constexpr bool kHoist = SM::kRows;                       // D <= 2: every per-thread index is tile-invariant
  constexpr int RG = NT / KH < K ? NT / KH : K;            // row groups of the copy-out
  constexpr int RPT = (K + RG - 1) / RG;                   // rows per thread of the copy-out
  constexpr int STRIDE = NC + 1, TABN = 2 * D * STRIDE;    // CG then CA, contiguous per tile
  static_assert(G * D * NC <= 96 && 192 + G * NC <= NT && G * 5 * (1 << D) <= NT, "role layout");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);
  const int tid = threadIdx.x;

  // ---- once per CTA: facts per (kind, signature) -----------------------------------------------------
  for (int x = tid; x < 2 * K; x += NT) {
    const int kind = x / K, j = x % K;
    int dig[D], r = j;
#pragma unroll
    for (int d = D - 1; d >= 0; --d) { dig[d] = r % 6; r /= 6; }
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
    si.cfgW = cw; si.cfgO = co; si.valid = valid; si.rowsplit = rs; si.colsplit = cs;
    sm.sig[kind][j] = si;
  }
  for (int x = tid; x < G * D; x += NT) { sm.t[x / D].CG[x % D][NC] = 0; sm.t[x / D].CA[x % D][NC] = 0; }
  __syncthreads();

  // ---- tile-invariant roles of this thread ---------------------------------------------------------------
  int slot[3 * D];                                         // step 3: the table entries summing to R[tid]
  int partner = 0;                                         // step 4: index of R[dual b][dual a]
  int cp_a[RPT];                                           // step 5: a_idx * (NS+1) of row r + k * RG for both producer kinds
  int cp_b = 0;                                            // step 5: b_idx of columns 2jp, 2jp+1 for both consumer kinds
  const int cp_r = tid / KH, cp_jp = tid % KH;
  if (kHoist) {
    if (tid < NS * NS) {
      r_slots<D>(tid / NS, tid % NS, slot);
      partner = dual_vec<D>(tid % NS) * NS + dual_vec<D>(tid / NS);
    }
#pragma unroll
    for (int k = 0; k < RPT; ++k) {
      const int i = cp_r + k * RG;
      if (cp_r < RG && i < K) {
        const int a0 = sm.sig[0][i].a_idx, a1 = sm.sig[1][i].a_idx;       // a = NS (invalid) selects the zero row
        cp_a[k] = (a0 * (NS + 1)) | (a1 * (NS + 1)) << 16;
      } else {
        cp_a[k] = 0;
      }
    }
    if (cp_r < RG) {
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int b = sm.sig[q >> 1][2 * cp_jp + (q & 1)].b_idx;
        cp_b |= (b >= 0 ? b : NS) << (8 * q);                  // b = NS (invalid) selects the zero column
      }
    }
    for (int x = tid; x < G * (NS + 1) * (NS + 1); x += NT) sm.t[x / ((NS + 1) * (NS + 1))].Esym[x % ((NS + 1) * (NS + 1))] = 0;
  }
  // step 1 role: (tile in group, extent, level subset); step 2 roles: A [0,96) B [96,192) C [192,..)
  const int q_t = tid / (5 << D), q_x = (tid % (5 << D)) >> D, q_m = tid & ((1 << D) - 1);
  const int role_base = tid < 96 ? 0 : (tid < 192 ? 96 : 192);
  const int role_i = tid - role_base;
  const int role_t = role_base == 192 ? role_i / NC : role_i / (D * NC);      // tile in group
  const int role_d = (role_i % (D * NC)) / NC;                                // level (roles A, B)
  const int role_cfg = role_i % NC;
  int role_m0 = 0, role_m1 = 0;
  cfg_masks<D>(role_cfg, role_m0, role_m1);
  const int64_t cap_layer = mp.mem_cap / L;
  const int ngroups = (ntiles + G - 1) / G;

  int grp = blockIdx.x;
  if (grp >= ngroups) return;
  int l0 = (int)(((int64_t)grp * G) % L);                  // layer index of the group's first tile
  const int l_step = (int)(((int64_t)gridDim.x * G) % L);
  int buf = 0;
  // records: thread 5*t + part stages 16-byte part (or the previous kind) of tile t of the group
  auto stage_group = [&](int b, int g, int lfirst) {
    if (tid < 5 * G) {
      const int t = tid / 5, part = tid % 5;
      int tile = g * G + t;
      if (tile >= ntiles) tile = ntiles - 1;                // ragged tail: restage a valid record, never used
      int l = lfirst + t;
      while (l >= L) l -= L;
      const autoddl_layer* cur = layers + tile;
      RecBuf* dst = &sm.rec[b][t];
      if (part < 4) cp_async16(reinterpret_cast<unsigned char*>(dst) + 16 * part, reinterpret_cast<const unsigned char*>(cur) + 16 * part);
      else cp_async4(&dst->kind_prev, &(l > 0 ? cur - 1 : cur)->kind);
    }
  };
  stage_group(0, grp, l0);
  cp_async_wait_all();
  __syncthreads();

  while (grp < ngroups) {
    const int grp_n = grp + gridDim.x;
    int l0_n = l0 + l_step;
    if (l0_n >= L) l0_n -= L;
    stage_group(buf ^ 1, grp_n < ngroups ? grp_n : grp, grp_n < ngroups ? l0_n : l0);
    const int tile0 = grp * G;
    const int nt = ntiles - tile0 < G ? ntiles - tile0 : G;   // tiles of this group that exist
    auto layer_of = [&](int t) { int l = l0 + t; while (l >= L) l -= L; return l; };
    int kinds = 0;                                           // (kind, kind_prev) of every tile of the group, read before
#pragma unroll                                               // the record buffer can be restaged by a faster thread
    for (int t = 0; t < G; ++t) kinds |= (sm.rec[buf][t].kind | sm.rec[buf][t].kind_prev << 1) << (2 * t);

    // ---- 1. Q[x][m]: x = M, Kd, N, in_rows, in_cols (the record's first five int64) ---------------------
    if (tid < G * (5 << D) && q_t < nt)
      sm.t[q_t].Q[q_x][q_m] = cdiv_magic(sm.rec[buf][q_t].X[q_x], (uint32_t)mp.sub[q_m], mp.magic_sub[q_m]);
    __syncthreads();

    // ---- 2. tables per level and split configuration -------------------------------------------------------
    if (role_t < nt) {
      typename SM::PerTile& pt = sm.t[role_t];
      const RecBuf& rec = sm.rec[buf][role_t];
      if (role_base == 0 && role_i < G * D * NC) {
        if (layer_of(role_t) > 0) {                          // input tensor: Table 2 rows 2 and 3
          const int d = role_d;
          const int64_t n = pt.Q[3][role_m0] * pt.Q[4][role_m1] * (int64_t)rec.eb;
          const int64_t p = mp.size[d];
          int64_t cg = 0, ca = 0;
          if (p > 1) {
            cg = (p - 1) * (mp.alpha[d] + cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d]);
            ca = (p - 1) * mp.alpha[d] + n * mp.beta[d];
          }
          pt.CG[d][role_cfg] = cg;
          pt.CA[d][role_cfg] = ca;
        }
      } else if (role_base == 96 && role_i < G * D * NC) {
        if (rec.kind == AUTODDL_GEMM) {                      // weight gradient: AllReduce row
          const int d = role_d;
          const int64_t n = pt.Q[1][role_m0] * pt.Q[2][role_m1] * (int64_t)rec.wgb;
          const int64_t p = mp.size[d];
          pt.WAR[d][role_cfg] =
              p > 1 ? (2 * p - 1) * mp.alpha[d] + 2 * (p - 1) * cdiv_magic(n, (uint32_t)p, mp.magic_size[d]) * mp.beta[d] : 0;
        }
      } else if (role_base == 192 && role_i < G * NC) {
        pt.locW[role_cfg] = pt.Q[1][role_m0] * pt.Q[2][role_m1];
        pt.locO[role_cfg] = pt.Q[0][role_m0] * pt.Q[2][role_m1];
      }
    }
    __syncthreads();

    // ---- 3. VP[j] (node cost + penalty) and R[a][b] ------------------------------------------------------------
    for (int x = tid; x < nt * K; x += NT) {
      const int t = x / K, j = x % K;
      typename SM::PerTile& pt = sm.t[t];
      const RecBuf& rec = sm.rec[buf][t];
      const SigInfo si = sm.sig[rec.kind][j];
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
      const bool ok = si.valid && si.rowsplit <= rec.maxr && si.colsplit <= rec.maxc && (mp.mem_cap == 0 || mem <= cap_layer);
      pt.VP[j] = v + (ok ? 0 : AUTODDL_PEN);
      const size_t o = (size_t)(tile0 + t) * K + j;
      if (node) node[o] = v;
      if (mask) mask[o] = ok ? 1 : 0;
    }
    if (kHoist) {
      if (tid < NS * NS) {
#pragma unroll
        for (int t = 0; t < G; ++t) {
          if (t < nt && layer_of(t) > 0) {
            const int64_t* tab = &sm.t[t].CG[0][0];
            int64_t c = 0;
#pragma unroll
            for (int k = 0; k < 3 * D; ++k) c += tab[slot[k]];
            sm.t[t].E[tid] = c;
          }
        }
      }
    } else {
      if (layer_of(0) > 0) {
        const int64_t* tab = &sm.t[0].CG[0][0];
        for (int e = tid; e < NS * NS; e += NT) {
          int idx[3 * D];
          r_slots<D>(e / NS, e % NS, idx);
          int64_t c = 0;
#pragma unroll
          for (int k = 0; k < 3 * D; ++k) c += tab[idx[k]];
          sm.t[0].E[e] = c;
        }
      }
    }
    __syncthreads();

    if (kHoist) {
      // ---- 4. Esym[a][b] = R[a][b] + R[dual b][dual a]: forward leg + backward leg ------------------------------
      if (tid < NS * NS) {
#pragma unroll
        for (int t = 0; t < G; ++t)
          if (t < nt && layer_of(t) > 0) sm.t[t].Esym[(tid / NS) * (NS + 1) + tid % NS] = sm.t[t].E[tid] + sm.t[t].E[partner];
      }
      if (tid < 5 * G) cp_async_wait_all();                // the next group's records have landed; the barrier publishes them
      __syncthreads();
      // ---- 5. K x K expansion: one gather + one add per cell, 16-byte streaming stores ---------------------------
      if (cp_r < RG) {
#pragma unroll
        for (int t = 0; t < G; ++t) {
          if (t < nt) {
            const typename SM::PerTile& pt = sm.t[t];
            const int kind = (kinds >> (2 * t)) & 1, kind_prev = (kinds >> (2 * t + 1)) & 1;
            const bool first = layer_of(t) == 0;
            int64_t* out = T + (size_t)(tile0 + t) * K * K;
            const longlong2 vp = *reinterpret_cast<const longlong2*>(&pt.VP[2 * cp_jp]);
            const int bb = cp_b >> (16 * kind);
            const int b0 = bb & 0xff, b1 = (bb >> 8) & 0xff;
#pragma unroll
            for (int k = 0; k < RPT; ++k) {
              if (cp_r + k * RG < K) {
                const int ao = first ? NS * (NS + 1) : ((cp_a[k] >> (16 * kind_prev)) & 0xffff);   // layer 0: zero row
                longlong2 v;
                v.x = vp.x + pt.Esym[ao + b0];
                v.y = vp.y + pt.Esym[ao + b1];
                __stcs(reinterpret_cast<longlong2*>(out + (size_t)(cp_r + k * RG) * K + 2 * cp_jp), v);
              }
            }
          }
        }
      }
    } else {
      const typename SM::PerTile& pt = sm.t[0];
      const RecBuf& rec = sm.rec[buf][0];
      const int l = layer_of(0);
      int64_t* out = T + (size_t)tile0 * K * K;
      for (int c = tid; c < K * KH; c += NT) {
        const int i = c / KH, j = (c % KH) * 2;
        longlong2 v = make_longlong2(pt.VP[j], pt.VP[j + 1]);
        if (l > 0) {
          const int a = sm.sig[rec.kind_prev][i].a_idx;
          if (a < NS) {
            const int da = dual_vec<D>(a);
            const SigInfo& s0 = sm.sig[rec.kind][j];
            const SigInfo& s1 = sm.sig[rec.kind][j + 1];
            if (s0.b_idx >= 0) v.x += pt.E[a * NS + s0.b_idx] + pt.E[s0.db_idx * NS + da];
            if (s1.b_idx >= 0) v.y += pt.E[a * NS + s1.b_idx] + pt.E[s1.db_idx * NS + da];
          }
        }
        __stcs(reinterpret_cast<longlong2*>(out + (size_t)i * K + j), v);
      }
      if (tid < 5 * G) cp_async_wait_all();
      __syncthreads();                                     // E is rewritten by the next group's step 3; publishes the records
    }
    grp = grp_n;
    l0 = l0_n;
    buf ^= 1;
  }
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
  const int per_sm = (D == 3) ? 1 : 3;
  const int ngroups = (ntiles + TileSmem<D>::G - 1) / TileSmem<D>::G;
  const int grid = ngroups < sms * per_sm ? ngroups : sms * per_sm;     // persistent, grid-stride over tile groups
  build_tables_kernel<D><<<grid, 256, smem, st>>>(d_layers, ntiles, L, mp, d_T, d_node, d_mask);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace

int launch_build_tables(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int64_t* d_T,
                        int64_t* d_node, uint8_t* d_mask, cudaStream_t st) {
  const int64_t nt = (int64_t)Bp * L;
  if (nt > 0x7fffffff) { set_error("Bp*L too large"); return AUTODDL_EINVAL; }
  switch (mp.ndim) {
    case 1: return launch_d<1>(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
    case 2: return launch_d<2>(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
    case 3: return launch_d<3>(d_layers, (int)nt, L, mp, d_T, d_node, d_mask, st);
  }
  set_error("ndim must be 1, 2 or 3");
  return AUTODDL_EINVAL;
}

}  // namespace autoddl
