// Shared host/device helpers of the CUDA path.  Nothing here is used by oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/autoddl.h"

namespace autoddl {

// ---- error plumbing (thread-local text, no exceptions across the ABI) ----------------------------
void set_error(const char* fmt, ...);
void clear_error();
void count_launch(int n = 1);

#define ADL_CUDA_CHECK(expr)                                                             \
  do {                                                                                   \
    cudaError_t _e = (expr);                                                             \
    if (_e != cudaSuccess) {                                                             \
      ::autoddl::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
      return AUTODDL_ECUDA;                                                              \
    }                                                                                    \
  } while (0)

// Debugging switches (they select between kernels that are all held to the same bit-exact parity) exist only in builds
// with -DAUTODDL_DEBUG_SWITCHES: the dispatch of the shipped library never depends on the caller's environment.
#ifdef AUTODDL_DEBUG_SWITCHES
#include <stdlib.h>
#define ADL_DEBUG_ENV(name) (getenv(name) != nullptr)
#define ADL_DEBUG_ENV_INT(name, dflt) (getenv(name) ? atoi(getenv(name)) : (dflt))
#else
#define ADL_DEBUG_ENV(name) false
#define ADL_DEBUG_ENV_INT(name, dflt) (dflt)
#endif

#define ADL_REQUIRE(cond, ...)                  \
  do {                                          \
    if (!(cond)) {                              \
      ::autoddl::set_error(__VA_ARGS__);        \
      return AUTODDL_EINVAL;                    \
    }                                           \
  } while (0)

// ---- mesh / net passed to kernels by value ----------------------------------------------------------
constexpr int kMaxLevels = AUTODDL_MAX_LEVELS;
constexpr int kTabLevels = 5;                              // the table-factorised builders handle up to five levels
struct MeshParams {
  int32_t ndim;
  int32_t K;            // signatures per layer: 6^ndim (ndim <= 3), product of the allowed-row counts (ndim = 4, 5; R26)
  int32_t size[kMaxLevels];
  int32_t allow[kMaxLevels];     // signature rows allowed on the level (bit g = row g), 0x3f = all six
  int64_t alpha[kMaxLevels];     // alpha of the level's link class
  int64_t beta[kMaxLevels];      // beta  of the level's link class
  int64_t mem_cap;      // 0 = none
  int64_t accum;        // micro-batches per mini-batch (>= 1): multiplies the redistribution costs
  int32_t sub[1 << kTabLevels];       // product of the sizes of the levels in subset m (bit e = level e), levels 0..4
  uint64_t magic_sub[1 << kTabLevels];   // ceil(2^64 / sub[m])
  uint64_t magic_size[kMaxLevels];  // ceil(2^64 / size[d])
  int32_t fold;                     // folded factorisation space (R28): groups of equal levels
  int32_t ngroups, gfirst[kMaxLevels], glen[kMaxLevels];
};

// fills *out (may be NULL); returns AUTODDL_OK or AUTODDL_EINVAL.  K of a valid mesh: mesh_num_sigs()
int validate_mesh_net(const autoddl_mesh* mesh, const autoddl_net* net, MeshParams* out);
int mesh_num_sigs(const autoddl_mesh* mesh);

// ---- kernel launchers (defined in the .cu files) ----------------------------------------------------
int launch_build_tables(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp,
                        int64_t* d_T, int64_t* d_node, uint8_t* d_mask, cudaStream_t st);
int launch_build_tables_folded(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp,
                               int64_t* d_T, int64_t* d_node, uint8_t* d_mask, cudaStream_t st);
bool fused_build_dp_supported(const MeshParams& mp, int32_t L);
size_t fused_bp_bytes(int32_t L);
int launch_build_dp_fused(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int64_t* d_T,
                          int64_t* d_node, uint8_t* d_mask, int64_t* d_opt_cost, int32_t* d_strategy, uint8_t* d_bp,
                          const int32_t* d_cd_init, int32_t S, int32_t* d_cd_s1, int32_t* d_cd_s2, cudaStream_t st);
bool fused_cd_sweep_supported(int32_t L, int32_t S);
int launch_chain_dp(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, uint8_t* d_bp,
                    int64_t* d_opt_cost, int32_t* d_strategy, cudaStream_t st);
bool chain_dp_cluster_supported(int32_t K, int32_t L);
int launch_chain_dp_cluster(const int64_t* d_T, int32_t Bp, int32_t L, int64_t* d_opt_cost, int32_t* d_strategy,
                            cudaStream_t st);
bool chain_dp_cluster_anyk_supported(int32_t K, int32_t L);
int launch_chain_dp_cluster_anyk(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, int64_t* d_opt_cost,
                                 int32_t* d_strategy, cudaStream_t st);
// resume: the first sweep (d_prev == NULL) or the first two sweeps (d_prev = the strategies after sweep 1) have been done
// already and their result is in d_strategy; continue from there
// sbp_rows: d_T was built by this library (identical rows per producer-signature class may be read through one row)
int launch_coord_descent(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, const int32_t* d_init,
                         int32_t S, int32_t max_sweeps, int64_t* d_cost, int32_t* d_strategy,
                         int32_t* d_sweeps, cudaStream_t st, bool resume = false, bool sbp_rows = false,
                         const int32_t* d_prev = nullptr);
// library-built tables of two / three mesh levels in factor form (factors.cu): the factors, the chain DP on them, and
// Coordinate Descent from many starts by best-response look-ups
bool factors_supported(const MeshParams& mp);
size_t factors_bytes(const MeshParams& mp, int32_t Bp, int32_t L);
int launch_build_factors(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int64_t* d_F, cudaStream_t st);
bool chain_dp_scan_supported(const MeshParams& mp, int32_t Bp, int32_t L);
size_t chain_dp_scan_bytes(const MeshParams& mp, int32_t Bp, int32_t L);
int launch_chain_dp_scan(const int64_t* d_F, int32_t Bp, int32_t L, const MeshParams& mp, void* d_work, int64_t* d_opt_cost,
                         int32_t* d_strategy, cudaStream_t st);
bool cd_lookup_tab_supported(int32_t K, int32_t L, int32_t S);
size_t cd_lookup_tab_workspace_bytes(int32_t K, int32_t Bp, int32_t L);
int launch_cd_lookup_tab(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, void* d_work, const int32_t* d_init, int32_t S,
                         int32_t max_sweeps, int64_t* d_cost, int32_t* d_strategy, int32_t* d_sweeps, cudaStream_t st);
bool chain_dp_scan_tab_supported(int32_t K, int32_t Bp, int32_t L);
size_t chain_dp_scan_tab_bytes(int32_t K, int32_t Bp, int32_t L);
int launch_chain_dp_scan_tab(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, void* d_work, int64_t* d_opt_cost,
                             int32_t* d_strategy, cudaStream_t st);
bool cd_lookup_supported(const MeshParams& mp, int32_t L, int32_t S);
size_t cd_lookup_workspace_bytes(const MeshParams& mp, int32_t Bp, int32_t L);
int launch_cd_lookup(const int64_t* d_F, int32_t Bp, int32_t L, const MeshParams& mp, void* d_work, const int32_t* d_init, int32_t S,
                     int32_t max_sweeps, int64_t* d_cost, int32_t* d_strategy, int32_t* d_sweeps, cudaStream_t st);
int launch_metropolis(const int64_t* d_T, int32_t Bp, int32_t L, int32_t K, const int32_t* d_init, int32_t S,
                      int32_t nsteps, int64_t tau_ps, uint64_t seed, int64_t* d_best_cost, int32_t* d_best_strategy,
                      int64_t* d_final_cost, int32_t* d_final_strategy, int32_t* d_accepted, cudaStream_t st);
size_t fit_workspace_bytes();
int launch_fit_alpha_beta(const int32_t* d_kind, const int32_t* d_p, const int64_t* d_bytes, const double* d_time,
                          int64_t N, double* d_out, double* d_work, cudaStream_t st);
int launch_copy_probe(const void* src, void* dst, size_t bytes, cudaStream_t st);
int launch_best_of_starts(const int64_t* d_cost, int32_t Bp, int32_t S, int64_t* d_best_cost, int32_t* d_best_start,
                          cudaStream_t st);
int launch_segment_optima(const int64_t* d_T, const int64_t* d_node, const uint8_t* d_mask, int32_t L, int32_t K,
                          int64_t* d_tri, cudaStream_t st);
int launch_stage_transfer(const autoddl_layer* d_layers, int32_t L, int64_t q, int64_t m, int64_t alpha, int64_t beta,
                          int64_t* d_xfer, cudaStream_t st);
size_t partition_workspace_bytes(int32_t L, int32_t stages);
int launch_partition(const int64_t* d_tri, const int64_t* d_xfer, int32_t L, int32_t stages, int32_t objective, void* d_work,
                     int64_t* d_value, int32_t* d_cuts, cudaStream_t st);
int launch_segment_strategies(const int64_t* d_T, const int64_t* d_node, const uint8_t* d_mask, int32_t L, int32_t K,
                              const int32_t* d_cuts, int32_t stages, uint8_t* d_bp, int64_t* d_seg_cost, int32_t* d_strategy,
                              cudaStream_t st);
int launch_store_probe(int64_t* d_T, int32_t Bp, int32_t L, int32_t cells, cudaStream_t st);
int device_sm_count();                                     // multiprocessors of the current device (148 if the query fails)

// ---- device helpers ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
// TMA 1-D bulk copy global -> shared, completion signalled on an mbarrier (bytes % 16 == 0, 16-B aligned)
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar,
                                         uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
      ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}

}  // namespace autoddl
