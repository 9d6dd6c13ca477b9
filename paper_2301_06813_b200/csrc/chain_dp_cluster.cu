// (a2) chain DP for ONE long chain with K = 216 spread over a thread-block cluster.
//
// A single chain is sequential in the layer index, so one CTA cannot stream a 373 KB tile per step at more than
// a few per cent of HBM speed.  Here a cluster of 8 CTAs (8 SMs) shares every step:
//   - CTA r owns rows i in [27 r, 27 r + 27) of every tile: one contiguous 46,656-byte block per layer, streamed
//     through a 4-stage ring by TMA bulk copies (cp.async.bulk + mbarrier complete_tx);
//   - thread j < 216 scans its column over the CTA's 27 rows in ascending i (strict '<': smallest index wins)
//     with f read from the CTA's own 27-entry slice of f_{l-1};
//   - the partial (value, row) of column j goes straight into the shared memory of the CTA that owns column j
//     (j / 27) with st.async over DSMEM, which also completes the transaction count of that CTA's mbarrier;
//   - 8 lanes per owned column merge the 8 partials with three shuffle steps on (value, row) -- row blocks are
//     disjoint, so the smaller row wins ties -- and write f_l[27 q + c]: exactly the slice that CTA needs as
//     f_{l-1}[i] for its rows of the next tile.
// One reduce-scatter per layer and no all-gather, no cluster-wide barrier inside the layer loop.  Back-pointers
// stay in shared memory (27 per layer per CTA), are gathered into CTA 0 at the end and walked there.
// Results are identical to the definition (R9): every comparison is on (value, smallest row).
#include "common.cuh"

namespace autoddl {

namespace {

constexpr int CK = 216, CC = 8, CR = CK / CC;             // signatures, CTAs per cluster, rows (and owned columns) per CTA
constexpr int CSTAGES = 4;
constexpr int CSTAGE_BYTES = CR * CK * 8;                 // 46,656
constexpr int CNT = 256;                                  // warps 0..6: column threads (216 active); warp 7: producer
static_assert(CSTAGE_BYTES % 16 == 0, "bulk copy granularity");

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(const void* p, uint32_t rank) {
  uint32_t a = smem_u32(p), r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
  return r;
}
// 16-byte remote store that completes 16 bytes of the remote mbarrier's transaction count
__device__ __forceinline__ void st_async_v2(uint32_t remote_addr, int64_t a, int64_t b, uint32_t remote_mbar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
               ::"r"(remote_addr), "l"(a), "l"(b), "r"(remote_mbar) : "memory");
}
__device__ __forceinline__ void st_cluster_u8(uint32_t remote_addr, uint32_t v) {
  asm volatile("st.shared::cluster.u8 [%0], %1;" ::"r"(remote_addr), "r"(v) : "memory");
}
__device__ __forceinline__ void st_cluster_b64(uint32_t remote_addr, int64_t v) {
  asm volatile("st.shared::cluster.b64 [%0], %1;" ::"r"(remote_addr), "l"(v) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_cluster(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}

struct ClusterSmem {
  alignas(128) int64_t stage[CSTAGES][CR * CK];           // row blocks of the tiles in flight; reused for the gathered
                                                          // back-pointers [L][CK] (CTA 0) after the last layer
  alignas(16) int64_t slot[2][CC][CR][2];                 // [layer parity][source CTA][owned column] = (value, row)
  alignas(16) int64_t f[2][CR];                           // this CTA's slice of f, by layer parity
  alignas(16) int64_t ffinal[CK];                         // CTA 0: f_{L-1} of all columns
  alignas(8) uint64_t full[CSTAGES], empty[CSTAGES], recv[2];
};

__global__ void __cluster_dims__(CC, 1, 1) __launch_bounds__(CNT, 1)
chain_dp216_cluster_kernel(const int64_t* __restrict__ T, int L, int64_t* __restrict__ opt_cost,
                           int32_t* __restrict__ strategy) {
  extern __shared__ __align__(128) unsigned char smem_cl[];
  ClusterSmem& sm = *reinterpret_cast<ClusterSmem*>(smem_cl);
  uint8_t* bp = smem_cl + sizeof(ClusterSmem);             // [L][CR]: back-pointers of the columns this CTA owns
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t r = cluster_ctarank();
  const int p = blockIdx.x / CC;                           // one chain per cluster
  const int64_t* Tp = T + (size_t)p * L * CK * CK;

  if (tid == 0) {
    for (int s = 0; s < CSTAGES; ++s) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], 7); }
    mbar_init(&sm.recv[0], 1);
    mbar_init(&sm.recv[1], 1);
    mbar_fence_init();
  }
  if (tid < CR) sm.f[0][tid] = __ldg(Tp + CR * r + tid);   // f_0[j] = T[0][0][j] for the owned columns
  __syncthreads();
  cluster_sync_all();                                      // every CTA's mbarriers exist before any remote store

  if (tid >= 224) {
    // ================= producer warp: one lane streams this CTA's row blocks =================
    if (tid == 224) {
      const uint64_t pol = policy_evict_first();
      const unsigned char* src = reinterpret_cast<const unsigned char*>(Tp + (size_t)CK * CK + (size_t)CR * r * CK);
      for (int b = 0; b < L - 1; ++b) {
        const int s = b % CSTAGES;
        if (b >= CSTAGES) mbar_wait(&sm.empty[s], ((b / CSTAGES) - 1) & 1);
        mbar_arrive_expect_tx(&sm.full[s], CSTAGE_BYTES);
        bulk_g2s(sm.stage[s], src + (size_t)b * CK * CK * 8, CSTAGE_BYTES, &sm.full[s], pol);
      }
    }
  } else {
    // ================= column threads =================
    const int j = tid;                                     // column (tid < 216)
    const bool col = j < CK;
    const uint32_t owner = col ? j / CR : 0;
    for (int l = 1; l < L; ++l) {
      const int b = l - 1, s = b % CSTAGES, par = l & 1;
      if (tid == 0) mbar_arrive_expect_tx(&sm.recv[par], CC * CR * 16);     // this layer's 8 x 27 partials
      mbar_wait(&sm.full[s], (b / CSTAGES) & 1);
      if (col) {
        const int64_t* tile = sm.stage[s] + j;
        const int64_t* f = sm.f[par ^ 1];
        int64_t best = INT64_MAX;
        int arg = 0;
        int64_t tv[CR];
#pragma unroll
        for (int k = 0; k < CR; ++k) tv[k] = tile[k * CK];  // all 27 rows in flight
#pragma unroll
        for (int k = 0; k < CR; ++k) {
          const int64_t v = f[k] + tv[k];
          if (v < best) { best = v; arg = k; }
        }
        st_async_v2(map_to_cta(&sm.slot[par][r][j - CR * owner][0], owner), best, (int64_t)(CR * r + arg),
                    map_to_cta(&sm.recv[par], owner));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.empty[s]);            // this warp is done with the stage
      {                                                    // 8 lanes per owned column merge the 8 row blocks
        while (!mbar_try_wait_cluster(&sm.recv[par], ((l - 1) >> 1) & 1)) {
        }
        const int mc = tid >> 3, mq = tid & 7;             // owned column (< 27 for tid < 216), source CTA
        const bool mine = tid < CR * CC;
        int64_t bv = mine ? sm.slot[par][mq][mc][0] : INT64_MAX;
        int64_t bi = mine ? sm.slot[par][mq][mc][1] : 0;
#pragma unroll
        for (int off = 1; off < 8; off <<= 1) {            // row blocks are disjoint: the smaller row wins ties
          const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
          const int64_t oi = __shfl_xor_sync(0xffffffffu, bi, off);
          if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if (mine && mq == 0) {
          sm.f[par][mc] = bv;
          bp[(size_t)l * CR + mc] = (uint8_t)bi;
        }
      }
      asm volatile("bar.sync 1, 224;" ::: "memory");       // f_l slice is complete for the next layer's scan
    }
  }

  // ---- gather f_{L-1} and all back-pointers into CTA 0, then walk back there --------------------------------
  __syncthreads();
  cluster_sync_all();                                      // every CTA has finished its last tile: stage memory is free
  {
    const int par = (L - 1) & 1;
    if (tid < CR) st_cluster_b64(map_to_cta(&sm.ffinal[CR * r + tid], 0), sm.f[par][tid]);
    uint8_t* gath = reinterpret_cast<uint8_t*>(sm.stage);  // CTA 0: [L][CK]
    for (int x = tid; x < L * CR; x += CNT) {
      const int l = x / CR, c = x % CR;
      st_cluster_u8(map_to_cta(gath + (size_t)l * CK + CR * r + c, 0), l >= 1 ? bp[x] : 0);
    }
  }
  cluster_sync_all();
  if (r == 0 && tid < 32) {
    const uint8_t* gath = reinterpret_cast<const uint8_t*>(sm.stage);
    int64_t bv = INT64_MAX;
    int bi = CK;
    for (int c = lane; c < CK; c += 32) {
      const int64_t v = sm.ffinal[c];
      if (v < bv) { bv = v; bi = c; }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if (lane == 0) {
      int32_t* sp = strategy + (size_t)p * L;
      opt_cost[p] = bv;
      int sidx = bi;
      sp[L - 1] = sidx;
      for (int l = L - 1; l >= 1; --l) {
        sidx = gath[(size_t)l * CK + sidx];
        sp[l - 1] = sidx;
      }
    }
  }
}

// ---- any K <= 256 (four / five mesh levels, R26): K = 81, 243 are odd, so a tile row is only 8-byte aligned and neither
// column pairs nor 16-byte-aligned row blocks exist.  The decomposition is the one above: CTA r owns the rows and the
// columns [CR r, CR r + CR) with CR = ceil(K / 8), the last CTAs may own fewer or none.  (Holding the row block in
// registers one layer ahead instead of staging it -- 8-byte loads coalesced over the columns -- was measured: 271 us on
// config 7 against 173 us for the kernel below; 1024 threads with four row groups per column: 384 us.)
constexpr int ACRMAX = 32;                                 // CR <= 32

// A row block [e0, e1) of an odd-K table starts and ends on 8-byte
// boundaries only, but the 16-byte-aligned span around it is a legal bulk copy: the copy starts one element early when e0
// is odd (the consumers read at offset `e0 & 1`) and stops one element short when e1 is odd -- that last element is
// fetched by the producer lane with a plain load and stored to shared memory before it arms the stage's mbarrier.
// Everything else is the K = 216 kernel.  KT = 0: K, CR and the CTA's row count are run-time values and every row access
// is predicated, which doubles the instruction count of the scan; KT > 0 (81, 243: the paper's rows on four / five
// levels): K = KT and CR = ACR are compile-time, and the CTAs that own fewer than CR rows keep the missing rows of every
// stage filled with 2^62 (never the minimum: cells are < 2^62 / L), so that all CTAs run the same unpredicated scan.
constexpr int TNT = 288;                                   // warps 0..7: column threads; warp 8: producer

struct ClusterTmaSmem {
  alignas(16) int64_t slot[2][CC][ACRMAX][2];
  alignas(16) int64_t f[2][ACRMAX];
  alignas(16) int64_t ffinal[256];
  alignas(8) uint64_t full[4], empty[4], recv[2];
};

template <int KT, int ACR>
__global__ void __cluster_dims__(CC, 1, 1) __launch_bounds__(TNT, 1)
chain_dp_cluster_tma_anyk_kernel(const int64_t* __restrict__ T, int L, int Krt, int nstages, int stage_elems, int gath_off,
                                 int64_t* __restrict__ opt_cost, int32_t* __restrict__ strategy) {
  extern __shared__ __align__(128) unsigned char smem_cl[];
  int64_t* stage0 = reinterpret_cast<int64_t*>(smem_cl);                         // [nstages][stage_elems]
  ClusterTmaSmem& sm = *reinterpret_cast<ClusterTmaSmem*>(smem_cl + (size_t)nstages * stage_elems * 8);
  uint8_t* bp = reinterpret_cast<uint8_t*>(&sm) + sizeof(ClusterTmaSmem);        // [L][ACRMAX]
  uint8_t* gath = smem_cl + gath_off;                      // CTA 0, after the last layer: [L][K], in the stage memory if it fits
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t r = cluster_ctarank();
  const int p = blockIdx.x / CC;
  constexpr bool EXACT = KT != 0;
  constexpr int64_t HUGE_COST = (int64_t)1 << 62;
  const int K = EXACT ? KT : Krt;
  const size_t pb = (size_t)p * L * K * K;                 // element index of the chain's first cell
  const int64_t* Tp = T + pb;
  const int CR = EXACT ? ACR : (K + CC - 1) / CC;
  const int r0 = CR * (int)r;
  const int nr = K - r0 < 0 ? 0 : (K - r0 < CR ? K - r0 : CR);

  if (tid == 0) {
    for (int s = 0; s < nstages; ++s) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], 8); }
    mbar_init(&sm.recv[0], 1);
    mbar_init(&sm.recv[1], 1);
    mbar_fence_init();
  }
  if (tid < 2 * ACRMAX) sm.f[tid / ACRMAX][tid % ACRMAX] = 0;
  if (EXACT && nr < CR)                                    // rows this CTA does not own: never the minimum
    for (int x = nr * K + tid; x < stage_elems; x += TNT)
      for (int s = 0; s < nstages; ++s) stage0[(size_t)s * stage_elems + x] = HUGE_COST;
  __syncthreads();
  if (tid < nr) sm.f[0][tid] = __ldg(Tp + r0 + tid);
  __syncthreads();
  cluster_sync_all();

  if (tid >= 256) {
    // ================= producer warp: one lane streams this CTA's row blocks =================
    if (tid == 256) {
      const uint64_t pol = policy_evict_first();
      for (int b = 0; b < L - 1; ++b) {
        const int s = b % nstages;
        if (b >= nstages) mbar_wait(&sm.empty[s], ((b / nstages) - 1) & 1);
        int64_t* dst = stage0 + (size_t)s * stage_elems;
        const size_t e0 = pb + ((size_t)(b + 1) * K + r0) * K, e1 = e0 + (size_t)nr * K;
        const size_t a0 = e0 & ~(size_t)1, a1 = e1 & ~(size_t)1;
        if ((e1 & 1) && nr > 0) dst[e1 - 1 - a0] = __ldcs(T + e1 - 1);           // the element past the aligned span
        if (EXACT && nr < CR) dst[e1 - a0] = HUGE_COST;    // first cell of the rows not owned (a copy with e0 odd ends there)
        const uint32_t bytes = nr > 0 ? (uint32_t)((a1 - a0) * 8) : 0u;
        mbar_arrive_expect_tx(&sm.full[s], bytes);
        if (bytes) bulk_g2s(dst, T + a0, bytes, &sm.full[s], pol);
      }
    }
  } else {
    // ================= column threads =================
    const int j = tid;
    const bool col = j < K;
    const uint32_t owner = col ? j / CR : 0;
    for (int l = 1; l < L; ++l) {
      const int b = l - 1, s = b % nstages, par = l & 1;
      if (tid == 0) mbar_arrive_expect_tx(&sm.recv[par], (uint32_t)(CC * nr * 16));
      mbar_wait(&sm.full[s], (b / nstages) & 1);
      if (col) {
        const size_t e0 = pb + ((size_t)l * K + r0) * K;
        const int64_t* tile = stage0 + (size_t)s * stage_elems + (e0 & 1) + j;
        const int64_t* f = sm.f[par ^ 1];
        int64_t best = INT64_MAX;
        int arg = 0;
        int64_t tv[ACR];
#pragma unroll
        for (int k = 0; k < ACR; ++k) tv[k] = (EXACT || k < nr) ? tile[k * K] : 0;
#pragma unroll
        for (int k = 0; k < ACR; ++k)
          if (EXACT || k < nr) {
            const int64_t v = f[k] + tv[k];
            if (v < best) { best = v; arg = k; }
          }
        st_async_v2(map_to_cta(&sm.slot[par][r][j - CR * (int)owner][0], owner), best, (int64_t)(r0 + arg),
                    map_to_cta(&sm.recv[par], owner));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.empty[s]);
      if (nr > 0) {
        while (!mbar_try_wait_cluster(&sm.recv[par], ((l - 1) >> 1) & 1)) {
        }
      }
      {
        const int mc = tid >> 3, mq = tid & 7;
        const bool mine = mc < nr;
        int64_t bv = mine ? sm.slot[par][mq][mc][0] : INT64_MAX;
        int64_t bi = mine ? sm.slot[par][mq][mc][1] : 0;
#pragma unroll
        for (int off = 1; off < 8; off <<= 1) {
          const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
          const int64_t oi = __shfl_xor_sync(0xffffffffu, bi, off);
          if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if (mine && mq == 0) {
          sm.f[par][mc] = bv;
          bp[(size_t)l * ACRMAX + mc] = (uint8_t)bi;
        }
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");
    }
  }

  // ---- gather f_{L-1} and all back-pointers into CTA 0, then walk back there --------------------------------
  __syncthreads();
  cluster_sync_all();                                      // every CTA has finished its last tile: stage memory is free
  {
    const int par = (L - 1) & 1;
    if (tid < nr) st_cluster_b64(map_to_cta(&sm.ffinal[r0 + tid], 0), sm.f[par][tid]);
    for (int x = tid; x < L * ACRMAX; x += TNT) {
      const int l = x / ACRMAX, c = x % ACRMAX;
      if (c < nr) st_cluster_u8(map_to_cta(gath + (size_t)l * K + r0 + c, 0), l >= 1 ? bp[x] : 0);
    }
  }
  cluster_sync_all();
  if (r == 0 && tid < 32) {
    int64_t bv = INT64_MAX;
    int bi = K;
    for (int c = lane; c < K; c += 32) {
      const int64_t v = sm.ffinal[c];
      if (v < bv) { bv = v; bi = c; }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if (lane == 0) {
      int32_t* sp = strategy + (size_t)p * L;
      opt_cost[p] = bv;
      int sidx = bi;
      sp[L - 1] = sidx;
      for (int l = L - 1; l >= 1; --l) {
        sidx = gath[(size_t)l * K + sidx];
        sp[l - 1] = sidx;
      }
    }
  }
}

}  // namespace

// One cluster of 8 CTAs per chain.  Supported for K = 216 and L <= 864 (the gathered back-pointers must fit the
// stage memory of CTA 0); the caller falls back to the one-CTA kernel otherwise or if the launch is refused.
bool chain_dp_cluster_supported(int32_t K, int32_t L) { return K == CK && L >= 2 && (size_t)L * CK <= (size_t)CSTAGES * CSTAGE_BYTES; }

int launch_chain_dp_cluster(const int64_t* d_T, int32_t Bp, int32_t L, int64_t* d_opt_cost, int32_t* d_strategy,
                            cudaStream_t st) {
  const size_t smem = (sizeof(ClusterSmem) + (size_t)L * CR + 127) / 128 * 128;
  if (smem > 227 * 1024) { set_error("chain_dp (cluster): %zu bytes of shared memory needed", smem); return AUTODDL_EINVAL; }
  ADL_CUDA_CHECK(cudaFuncSetAttribute(chain_dp216_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  chain_dp216_cluster_kernel<<<Bp * CC, CNT, smem, st>>>(d_T, L, d_opt_cost, d_strategy);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

// stage = one row block plus the two elements of alignment slack, rounded to 16 bytes; the gathered back-pointers of
// CTA 0 reuse the stage memory when they fit there, else they get a region of their own
struct TmaAnyCfg { int nstages, stage_elems, gath_off; size_t smem; };
static bool tma_anyk_config(int32_t K, int32_t L, TmaAnyCfg* c) {
  const int CR = (K + CC - 1) / CC;
  const int se = (CR * K + 2 + 1) & ~1;
  for (int ns = 4; ns >= 2; --ns) {
    const size_t stages = (size_t)ns * se * 8;
    size_t b = stages + sizeof(ClusterTmaSmem) + (size_t)L * ACRMAX;
    int goff = 0;
    if ((size_t)L * K > stages) { goff = (int)((b + 15) / 16 * 16); b = goff + (size_t)L * K; }
    if (b <= 227 * 1024) { *c = {ns, se, goff, (b + 127) / 128 * 128}; return true; }
  }
  return false;
}

// any 64 <= K <= 256 (smaller K: the one-CTA kernels are as fast); L limited by the back-pointers gathered in CTA 0
bool chain_dp_cluster_anyk_supported(int32_t K, int32_t L) {
  TmaAnyCfg c;
  return K >= 64 && K <= 256 && L >= 2 && tma_anyk_config(K, L, &c);
}

int launch_chain_dp_cluster_anyk(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, int64_t* d_opt_cost,
                                 int32_t* d_strategy, cudaStream_t st) {
  TmaAnyCfg c;
  if (!tma_anyk_config(K, L, &c)) { set_error("chain_dp (cluster): K = %d, L = %d does not fit shared memory", K, L); return AUTODDL_EINVAL; }
  const int CRk = (K + CC - 1) / CC;
  auto kern = K == 243 ? chain_dp_cluster_tma_anyk_kernel<243, 31> : K == 81 ? chain_dp_cluster_tma_anyk_kernel<81, 11>
            : CRk <= 8 ? chain_dp_cluster_tma_anyk_kernel<0, 8> : CRk <= 16 ? chain_dp_cluster_tma_anyk_kernel<0, 16>
            : CRk <= 24 ? chain_dp_cluster_tma_anyk_kernel<0, 24> : chain_dp_cluster_tma_anyk_kernel<0, 32>;
  ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem));
  kern<<<Bp * CC, TNT, c.smem, st>>>(d_T, L, K, c.nstages, c.stage_elems, c.gath_off, d_opt_cost, d_strategy);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
