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

// ---- any K <= 256 (four / five mesh levels, R26: K = 81, 243 are odd, so neither 16-byte-aligned TMA row blocks nor
// column pairs exist).  Same decomposition over a cluster of 8 CTAs -- CTA r owns the rows and the columns
// [CR r, CR r + CR) with CR = ceil(K / 8), the last CTAs may own fewer or none -- but the row block of a layer goes
// from global memory straight into registers: thread j holds its column's <= 32 rows of layer l + 1 (8-byte loads,
// coalesced over j, issued one layer ahead so that their latency hides behind layer l's exchange).  (1024 threads with
// four row groups per column and a warp-wide merge of 32 partials was measured: 271 -> 384 us on config 7.)
constexpr int ACRMAX = 32, ANT = 256;                   // the kernel is instantiated for ACR = 8, 16, 24, 32 >= CR

struct ClusterAnySmem {
  alignas(16) int64_t slot[2][CC][ACRMAX][2];              // [layer parity][source CTA][owned column] = (value, row)
  alignas(16) int64_t f[2][ACRMAX];
  alignas(16) int64_t ffinal[256];
  alignas(8) uint64_t recv[2];
};

template <int ACR>
__global__ void __cluster_dims__(CC, 1, 1) __launch_bounds__(ANT, 1)
chain_dp_cluster_anyk_kernel(const int64_t* __restrict__ T, int L, int K, int64_t* __restrict__ opt_cost,
                             int32_t* __restrict__ strategy) {
  extern __shared__ __align__(128) unsigned char smem_cl[];
  ClusterAnySmem& sm = *reinterpret_cast<ClusterAnySmem*>(smem_cl);
  uint8_t* bp = smem_cl + sizeof(ClusterAnySmem);          // [L][ACRMAX]: back-pointers of the columns this CTA owns
  uint8_t* gath = bp + (size_t)L * ACRMAX;                 // CTA 0: [L][K] gathered back-pointers
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t r = cluster_ctarank();
  const int p = blockIdx.x / CC;
  const int64_t* Tp = T + (size_t)p * L * K * K;
  const int CR = (K + CC - 1) / CC;
  const int r0 = CR * (int)r;
  const int nr = K - r0 < 0 ? 0 : (K - r0 < CR ? K - r0 : CR);      // rows = owned columns of this CTA

  if (tid == 0) {
    mbar_init(&sm.recv[0], 1);
    mbar_init(&sm.recv[1], 1);
    mbar_fence_init();
  }
  if (tid < nr) sm.f[0][tid] = __ldg(Tp + r0 + tid);       // f_0[j] = T[0][0][j] for the owned columns
  __syncthreads();
  cluster_sync_all();                                      // every CTA's mbarriers exist before any remote store

  const int j = tid;                                       // column
  const bool col = j < K;
  const uint32_t owner = col ? j / CR : 0;
  int64_t tn[ACR];                                         // this column's rows of the NEXT layer
  const int nrc = col ? nr : 0;
  const int64_t* next = Tp + ((size_t)K + r0) * K + j;     // row r0 of layer 1, column j
  auto load_rows = [&]() {
    const int64_t* src = next;
#pragma unroll
    for (int k = 0; k < ACR; ++k) {
      tn[k] = k < nrc ? __ldcs(src) : 0;
      src += K;
    }
    next += (size_t)K * K;
  };
  if (L > 1) load_rows();
  for (int l = 1; l < L; ++l) {
    const int par = l & 1;
    if (tid == 0) mbar_arrive_expect_tx(&sm.recv[par], (uint32_t)(CC * nr * 16));   // this layer's 8 x nr partials
    int64_t tv[ACR];
#pragma unroll
    for (int k = 0; k < ACR; ++k) tv[k] = tn[k];
    if (l + 1 < L) load_rows();                            // in flight during this layer's scan and exchange
    if (col) {
      const int64_t* f = sm.f[par ^ 1];
      int64_t best = INT64_MAX;
      int arg = 0;
#pragma unroll
      for (int k = 0; k < ACR; ++k)
        if (k < nr) {
          const int64_t v = f[k] + tv[k];
          if (v < best) { best = v; arg = k; }
        }
      st_async_v2(map_to_cta(&sm.slot[par][r][j - CR * (int)owner][0], owner), best, (int64_t)(r0 + arg),
                  map_to_cta(&sm.recv[par], owner));
    }
    if (nr > 0) {
      while (!mbar_try_wait_cluster(&sm.recv[par], ((l - 1) >> 1) & 1)) {
      }
    }
    {                                                      // 8 lanes per owned column merge the 8 row blocks
      const int mc = tid >> 3, mq = tid & 7;
      const bool mine = mc < nr;
      int64_t bv = mine ? sm.slot[par][mq][mc][0] : INT64_MAX;
      int64_t bi = mine ? sm.slot[par][mq][mc][1] : 0;
#pragma unroll
      for (int off = 1; off < 8; off <<= 1) {              // row blocks are disjoint: the smaller row wins ties
        const int64_t ov = __shfl_xor_sync(0xffffffffu, bv, off);
        const int64_t oi = __shfl_xor_sync(0xffffffffu, bi, off);
        if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
      }
      if (mine && mq == 0) {
        sm.f[par][mc] = bv;
        bp[(size_t)l * ACRMAX + mc] = (uint8_t)bi;
      }
    }
    __syncthreads();                                       // f_l slice is complete for the next layer's scan
  }

  // ---- gather f_{L-1} and all back-pointers into CTA 0, then walk back there --------------------------------
  cluster_sync_all();
  {
    const int par = (L - 1) & 1;
    if (tid < nr) st_cluster_b64(map_to_cta(&sm.ffinal[r0 + tid], 0), sm.f[par][tid]);
    for (int x = tid; x < L * ACRMAX; x += ANT) {
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

static size_t cluster_anyk_smem(int32_t K, int32_t L) {
  return (sizeof(ClusterAnySmem) + (size_t)L * ACRMAX + (size_t)L * K + 127) / 128 * 128;
}
// any 64 <= K <= 256: row blocks through registers; L limited by the back-pointers gathered in CTA 0
bool chain_dp_cluster_anyk_supported(int32_t K, int32_t L) {
  return K >= 64 && K <= 256 && L >= 2 && cluster_anyk_smem(K, L) <= 200 * 1024;
}

int launch_chain_dp_cluster_anyk(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, int64_t* d_opt_cost,
                                 int32_t* d_strategy, cudaStream_t st) {
  const size_t smem = cluster_anyk_smem(K, L);
  const int CRk = (K + CC - 1) / CC;
  auto kern = CRk <= 8 ? chain_dp_cluster_anyk_kernel<8> : CRk <= 16 ? chain_dp_cluster_anyk_kernel<16>
            : CRk <= 24 ? chain_dp_cluster_anyk_kernel<24> : chain_dp_cluster_anyk_kernel<32>;
  ADL_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<Bp * CC, ANT, smem, st>>>(d_T, L, K, d_opt_cost, d_strategy);
  count_launch();
  ADL_CUDA_CHECK(cudaGetLastError());
  return AUTODDL_OK;
}

}  // namespace autoddl
