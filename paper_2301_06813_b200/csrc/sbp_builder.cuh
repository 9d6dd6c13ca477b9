// Device-side pieces shared by the table builders (build_tables.cu) and the fused per-chain kernel (fused_chain.cu):
// signature rows, the per-level walk of a redistribution, magic-number division, per-signature facts.
// Everything has internal linkage (anonymous namespace): each translation unit gets its own copy.
#pragma once

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
// four / five levels (R26): the signature index runs over the allowed rows only; K is a launch parameter <= 256
template <> struct Pow<4> { static constexpr int K = 256, NS = 256, NC = 81; };
template <> struct Pow<5> { static constexpr int K = 256, NS = 1024, NC = 243; };

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
  uint8_t allowed;    // every per-level row of the signature is in the level's allowed set (mesh.link bits 8..13)
  int32_t rowsplit, colsplit;
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
__device__ __forceinline__ void r_slots(int av, int bv, int (&idx)[3 * D], const uint32_t* walk = c_walk.w) {
  constexpr int NC = Pow<D>::NC, STRIDE = NC + 1, CA_OFF = D * STRIDE, ZERO = NC;
  int c0[D], c1[D], c2[D], c3[D];
  bool r1[D], r2[D], r3[D];
  int pw = 1;
#pragma unroll
  for (int d = 0; d < D; ++d) {
    const int sh = 2 * (D - 1 - d);
    const uint32_t w = walk[((av >> sh) & 3) * 4 + ((bv >> sh) & 3)];
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

// facts per (layer kind, signature), built once per CTA
template <int D>
__device__ __forceinline__ void fill_sig_table(SigInfo (*sig)[Pow<D>::K], const MeshParams& mp, int tid, int nthreads) {
  constexpr int K = Pow<D>::K, NS = Pow<D>::NS;
  for (int x = tid; x < 2 * K; x += nthreads) {
    const int kind = x / K, j = x % K;
    int dig[D], r = j;
#pragma unroll
    for (int d = D - 1; d >= 0; --d) { dig[d] = r % 6; r /= 6; }
    SigInfo si{};
    int a = 0, b = 0, cw = 0, co = 0, pw = 1, rs = 1, cs = 1;
    bool valid = true, allowed = true;
#pragma unroll
    for (int d = 0; d < D; ++d) {
      const int g = dig[d];
      allowed = allowed && ((mp.allow[d] >> g) & 1);
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
    si.cfgW = cw; si.cfgO = co; si.valid = valid; si.allowed = allowed; si.rowsplit = rs; si.colsplit = cs;
    sig[kind][j] = si;
  }
}

}  // namespace

}  // namespace autoddl
