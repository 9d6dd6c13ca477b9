// (a1) SBP cost-table builder for sm_100a.
//
// T[p][l][i][j] = E(l,i,j) + V(l,j) + PEN*[j infeasible at l]      (R8)
//   E: forward + backward redistribution of layer l's input between producer-output signature i
//      and consumer-input signature j (collectives Table 2, PAPER.md:102-108;
//      link class per mesh level)
//   V: all-reduce of the weight gradient on every level where W is replicated
//   feasibility: split limits and per-device memory
//
// Design (differs from the plain per-cell evaluation on purpose):
//   one CTA builds one K x K tile.  A redistribution moves every mesh level through the fixed
//   state sequence  (start) -> after slice -> after reduce-scatter -> after all-to-all -> after
//   all-gather, and that sequence depends only on the level's own (from,to) pair; levels interact
//   only through the local tensor size at the moment a collective runs.  So per tile we compute
//     1. ceil(rows/f0), ceil(cols/f1) for every subset of levels               (<= 16 divisions)
//     2. CG[d][cfg], CA[d][cfg]: gather/scatter and all-to-all cost on level d when the levels are
//        split as cfg (3^D configurations)                                     (<= 81 divisions)
//     3. R[a][b] over the 4^D x 4^D state vectors: a sum of <= 3D table entries
//     4. E[a][b] = R[a][b] + R[dual b][dual a]   (in place: the map is an involution)
//     5. VP[j] = V + penalty, node, mask per consumer signature
//     6. the K x K expansion: one shared-memory gather + one 64-bit add per cell, 16-byte stores.
//   The kernel is then bound by the HBM write of 8 B per cell, not by integer arithmetic.
#include "common.cuh"

namespace autoddl {

namespace {

constexpr int kS0 = 0, kS1 = 1, kB = 2, kP = 3;

// per-level signature rows (PAPER.md:193 rows 0..2; replicate; partial pass-through), R1
__device__ __constant__ int8_t c_gemm_I[6] = {kS0, kB, kS1, kB, kP, kB};
__device__ __constant__ int8_t c_gemm_W[6] = {kB, kS1, kS0, kB, kB, kP};
__device__ __constant__ int8_t c_gemm_O[6] = {kS0, kS1, kP, kB, kP, kP};
__device__ __constant__ int8_t c_attn_IO[6] = {kS0, kS1, -1, kB, -1, -1};

__device__ __forceinline__ int64_t cdiv64(int64_t a, int64_t b) {
  // operands are non-negative; most values fit 32 bits, where the division is ~5x cheaper
  if (((uint64_t)a | (uint64_t)b) >> 32) return (a + b - 1) / b;
  const uint32_t ua = (uint32_t)a, ub = (uint32_t)b;
  const uint32_t q = ua / ub;
  return (int64_t)(q + (q * ub != ua));
}

__device__ __forceinline__ int split_code(int s) { return s == kS0 ? 1 : (s == kS1 ? 2 : 0); }
__device__ __forceinline__ bool is_split(int s) { return s == kS0 || s == kS1; }
__device__ __forceinline__ int dual_of(int s) { return s == kB ? kP : (s == kP ? kB : s); }

template <int D> struct Pow { };
template <> struct Pow<1> { static constexpr int K = 6, NS = 4, NC = 3; };
template <> struct Pow<2> { static constexpr int K = 36, NS = 16, NC = 9; };
template <> struct Pow<3> { static constexpr int K = 216, NS = 64, NC = 27; };

template <int D>
struct TileSmem {
  int64_t rowc[8];                        // ceil(in_rows / prod of the levels in the subset)
  int64_t colc[8];
  int64_t CG[D][Pow<D>::NC];              // all-gather == reduce-scatter cost on level d under split config
  int64_t CA[D][Pow<D>::NC];              // all-to-all cost
  int64_t VP[Pow<D>::K];                  // node cost + penalty per consumer signature
  int16_t aidx[Pow<D>::K];                // producer signature -> O state-vector index (or -1)
  int16_t bidx[Pow<D>::K];                // consumer signature -> I state-vector index (or -1)
  int64_t E[Pow<D>::NS * Pow<D>::NS];     // R, then E in place
};

template <int D>
__global__ void __launch_bounds__(256) build_tables_kernel(const autoddl_layer* __restrict__ layers, int ntiles,
                                                           int L, MeshParams mp, int64_t* __restrict__ T,
                                                           int64_t* __restrict__ node, uint8_t* __restrict__ mask) {
  constexpr int K = Pow<D>::K, NS = Pow<D>::NS, NC = Pow<D>::NC;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileSmem<D>& sm = *reinterpret_cast<TileSmem<D>*>(smem_raw);
  const int tid = threadIdx.x, NT = blockDim.x;

  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int l = tile % L;
    const autoddl_layer* cur = layers + tile;
    // uniform per CTA: served by one broadcast transaction each
    const int64_t in_rows = __ldg(&cur->in_rows), in_cols = __ldg(&cur->in_cols);
    const int kind = __ldg(&cur->kind);
    const int64_t eb = __ldg(&cur->act_bytes);
    const int kind_prev = (l > 0) ? __ldg(&(cur - 1)->kind) : AUTODDL_GEMM;

    // ---- 1. subset quotients ------------------------------------------------------------------
    if (tid < 2 * (1 << D)) {
      const int m = tid & ((1 << D) - 1);
      int64_t f = 1;
#pragma unroll
      for (int d = 0; d < D; ++d)
        if (m >> d & 1) f *= mp.size[d];
      if (tid < (1 << D)) sm.rowc[m] = cdiv64(in_rows, f);
      else                sm.colc[m] = cdiv64(in_cols, f);
    }
    // signature -> state-vector indices (base 4, level 0 most significant)
    for (int j = tid; j < K; j += NT) {
      int a = 0, b = 0, r = j;
      bool va = true, vb = true;
      int dig[D];
#pragma unroll
      for (int d = D - 1; d >= 0; --d) { dig[d] = r % 6; r /= 6; }
#pragma unroll
      for (int d = 0; d < D; ++d) {
        const int g = dig[d];
        int so, si;
        if (kind_prev == AUTODDL_GEMM) so = c_gemm_O[g]; else { so = c_attn_IO[g]; if (so < 0) { va = false; so = 0; } }
        if (kind == AUTODDL_GEMM) si = c_gemm_I[g]; else { si = c_attn_IO[g]; if (si < 0) { vb = false; si = 0; } }
        a = a * 4 + so;
        b = b * 4 + si;
      }
      sm.aidx[j] = va ? (int16_t)a : (int16_t)-1;
      sm.bidx[j] = vb ? (int16_t)b : (int16_t)-1;
    }
    __syncthreads();

    // ---- 2. collective costs per level and split configuration ----------------------------------
    if (l > 0 && tid < D * NC) {
      const int d = tid / NC, cfg = tid % NC;
      int m0 = 0, m1 = 0, r = cfg;
#pragma unroll
      for (int e = 0; e < D; ++e) {
        const int sp = r % 3; r /= 3;
        if (sp == 1) m0 |= 1 << e;
        if (sp == 2) m1 |= 1 << e;
      }
      const int64_t n = sm.rowc[m0] * sm.colc[m1] * eb;          // bytes of the local tensor
      const int64_t p = mp.size[d];
      int64_t cg = 0, ca = 0;
      if (p > 1) {                                                // Table 2
        cg = (p - 1) * (mp.alpha[d] + cdiv64(n, p) * mp.beta[d]);
        ca = (p - 1) * mp.alpha[d] + n * mp.beta[d];
      }
      sm.CG[d][cfg] = cg;
      sm.CA[d][cfg] = ca;
    }

    // ---- 5. per consumer signature: node cost, feasibility (independent of steps 2-4) -------------
    {
      const int64_t Mo = __ldg(&cur->M), Kd = __ldg(&cur->Kd), No = __ldg(&cur->N);
      const int64_t wgb = __ldg(&cur->wgrad_bytes), wsb = __ldg(&cur->wstate_bytes);
      const int64_t maxr = __ldg(&cur->max_split_rows), maxc = __ldg(&cur->max_split_cols);
      for (int j = tid; j < K; j += NT) {
        int dig[D], r = j;
#pragma unroll
        for (int d = D - 1; d >= 0; --d) { dig[d] = r % 6; r /= 6; }
        bool valid = true;
        int mI0 = 0, mI1 = 0;                 // level subsets splitting I's rows / cols
        int64_t fW0 = 1, fW1 = 1, fO0 = 1, fO1 = 1, rowsplit = 1, colsplit = 1;
#pragma unroll
        for (int d = 0; d < D; ++d) {
          const int g = dig[d];
          const int64_t p = mp.size[d];
          int si, so, sw;
          if (kind == AUTODDL_GEMM) { si = c_gemm_I[g]; so = c_gemm_O[g]; sw = c_gemm_W[g]; }
          else { si = so = c_attn_IO[g]; sw = kB; if (si < 0) { valid = false; si = so = kB; } }
          if (si == kS0) mI0 |= 1 << d;
          if (si == kS1) mI1 |= 1 << d;
          if (so == kS0) fO0 *= p;
          if (so == kS1) { fO1 *= p; colsplit *= p; }
          if (sw == kS0) fW0 *= p;
          if (sw == kS1) fW1 *= p;
          if (si == kS0 || so == kS0) rowsplit *= p;
        }
        int64_t v = 0, mem = 0;
        if (valid) {
          if (kind == AUTODDL_GEMM) {
            const int64_t nw = cdiv64(Kd, fW0) * cdiv64(No, fW1);
            const int64_t nbytes = nw * wgb;
#pragma unroll
            for (int d = 0; d < D; ++d) {
              const int64_t p = mp.size[d];
              if (c_gemm_W[dig[d]] == kB && p > 1)               // AllReduce row of Table 2
                v += (2 * p - 1) * mp.alpha[d] + 2 * (p - 1) * cdiv64(nbytes, p) * mp.beta[d];
            }
            mem = nw * wsb;
          }
          mem += (sm.rowc[mI0] * sm.colc[mI1] + cdiv64(Mo, fO0) * cdiv64(No, fO1)) * eb;
        }
        const bool ok = valid && rowsplit <= maxr && colsplit <= maxc &&
                        (mp.mem_cap == 0 || mem <= mp.mem_cap / L);
        sm.VP[j] = v + (ok ? 0 : AUTODDL_PEN);
        if (node) node[(size_t)tile * K + j] = v;
        if (mask) mask[(size_t)tile * K + j] = ok ? 1 : 0;
      }
    }
    __syncthreads();

    if (l > 0) {
      // ---- 3. R[a][b]: every level walks slice -> reduce-scatter -> all-to-all -> all-gather -----
      for (int e = tid; e < NS * NS; e += NT) {
        const int av = e / NS, bv = e % NS;
        int pw3[D];
        int c0[D], c1[D], c2[D], c3[D];   // split codes after slice / reduce / all-to-all / gather, times 3^level
        bool act1[D], act2[D], act3[D];
        {
          int w = 1;
#pragma unroll
          for (int d = 0; d < D; ++d) { pw3[d] = w; w *= 3; }
        }
#pragma unroll
        for (int d = 0; d < D; ++d) {
          const int a = (av >> (2 * (D - 1 - d))) & 3, b = (bv >> (2 * (D - 1 - d))) & 3;
          const int s0 = (a == kB && is_split(b)) ? b : a;                 // keep own slice: free
          act1[d] = (s0 == kP && b != kP);                                 // partial -> split
          const int s1 = act1[d] ? (b == kB ? kS1 : b) : s0;
          act2[d] = is_split(s1) && is_split(b) && s1 != b;                // change of split axis
          const int s2 = act2[d] ? b : s1;
          act3[d] = is_split(s2) && b == kB;                               // split -> replicated
          const int s3 = act3[d] ? kB : s2;
          c0[d] = split_code(s0) * pw3[d];
          c1[d] = split_code(s1) * pw3[d];
          c2[d] = split_code(s2) * pw3[d];
          c3[d] = split_code(s3) * pw3[d];
        }
        int64_t cost = 0;
        // reduce-scatter, innermost level first; message = local tensor before the scatter
#pragma unroll
        for (int d = D - 1; d >= 0; --d) {
          int cfg = 0;
#pragma unroll
          for (int e2 = 0; e2 < D; ++e2) cfg += (e2 > d) ? c1[e2] : (e2 < d ? c0[e2] : 0);
          if (act1[d]) cost += sm.CG[d][cfg];
        }
        // all-to-all, innermost first; message = local tensor after the exchange
#pragma unroll
        for (int d = D - 1; d >= 0; --d) {
          int cfg = 0;
#pragma unroll
          for (int e2 = 0; e2 < D; ++e2) cfg += (e2 > d) ? c2[e2] : (e2 < d ? c1[e2] : c2[e2]);
          if (act2[d]) cost += sm.CA[d][cfg];
        }
        // all-gather, outermost first; message = local tensor after the gather
#pragma unroll
        for (int d = 0; d < D; ++d) {
          int cfg = 0;
#pragma unroll
          for (int e2 = 0; e2 < D; ++e2) cfg += (e2 < d) ? c3[e2] : (e2 > d ? c2[e2] : 0);
          if (act3[d]) cost += sm.CG[d][cfg];
        }
        sm.E[e] = cost;
      }
      __syncthreads();

      // ---- 4. E[a][b] = R[a][b] + R[dual b][dual a], in place ----------------------------------------
      for (int e = tid; e < NS * NS; e += NT) {
        const int av = e / NS, bv = e % NS;
        int da = 0, db = 0;
#pragma unroll
        for (int d = 0; d < D; ++d) {
          const int sh = 2 * (D - 1 - d);
          da |= dual_of((av >> sh) & 3) << sh;
          db |= dual_of((bv >> sh) & 3) << sh;
        }
        const int e2 = db * NS + da;                  // partner cell; (e2's partner is e)
        if (e <= e2) {
          const int64_t s = sm.E[e] + sm.E[e2];
          sm.E[e] = s;
          sm.E[e2] = s;
        }
      }
      __syncthreads();
    }

    // ---- 6. expansion to K x K, two cells (16 bytes) per store -----------------------------------------
    {
      int64_t* out = T + (size_t)tile * K * K;
      constexpr int KH = K / 2;
      for (int c = tid; c < K * KH; c += NT) {
        const int i = c / KH, j = (c % KH) * 2;
        longlong2 v;
        v.x = sm.VP[j];
        v.y = sm.VP[j + 1];
        if (l > 0) {
          const int a = sm.aidx[i], b0 = sm.bidx[j], b1 = sm.bidx[j + 1];
          if (a >= 0 && b0 >= 0) v.x += sm.E[a * NS + b0];
          if (a >= 0 && b1 >= 0) v.y += sm.E[a * NS + b1];
        }
        __stcs(reinterpret_cast<longlong2*>(out + (size_t)i * K + j), v);
      }
    }
    __syncthreads();      // smem is reused by the next tile
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
  const int per_sm = (D == 3) ? 2 : 8;
  const int grid = ntiles < sms * per_sm ? ntiles : sms * per_sm;       // persistent, grid-stride over tiles
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
