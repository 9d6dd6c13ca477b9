// C-ABI entry points (include/autoddl.h): argument validation, workspace carving, launches.
#include <stdarg.h>
#include <string.h>

#include "common.cuh"

namespace autoddl {

static thread_local char g_err[512] = "";
static thread_local int64_t g_launches = 0;
static thread_local cudaEvent_t g_mark = nullptr;          // autoddl_profile_mark: one-shot event between the kernels of a search
static thread_local cudaEvent_t g_dp_done = nullptr;       // autoddl_search_host: one-shot event after tables + DP (same place)

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
void clear_error() { g_err[0] = 0; }
void count_launch(int n) { g_launches += n; }

static inline bool mesh_folded(const autoddl_mesh* mesh) { return (mesh->link[0] & AUTODDL_FOLD) != 0; }

// R28: groups = maximal runs of consecutive levels with equal size and link class
static int fold_groups(const autoddl_mesh* mesh, int32_t* first, int32_t* len) {
  int ng = 0;
  for (int d = 0; d < mesh->ndim; ++d) {
    if (d > 0 && mesh->size[d] == mesh->size[d - 1] && ((mesh->link[d] ^ mesh->link[d - 1]) & 1) == 0) {
      ++len[ng - 1];
    } else {
      first[ng] = d;
      len[ng++] = 1;
    }
  }
  return ng;
}

int validate_mesh_net(const autoddl_mesh* mesh, const autoddl_net* net, MeshParams* out) {
  ADL_REQUIRE(mesh != nullptr, "mesh is NULL");
  ADL_REQUIRE(mesh->ndim >= 1 && mesh->ndim <= kMaxLevels, "mesh.ndim = %d, must be 1..%d", mesh->ndim, kMaxLevels);
  const bool fold = mesh_folded(mesh);
  ADL_REQUIRE(fold || mesh->ndim <= kTabLevels, "mesh.ndim = %d: more than %d levels exist only in the folded space "
              "(AUTODDL_FOLD in mesh.link[0])", mesh->ndim, kTabLevels);
  for (int d = 0; d < mesh->ndim; ++d) {
    ADL_REQUIRE(mesh->size[d] >= 1 && mesh->size[d] <= 65536, "mesh.size[%d] = %d out of range", d, mesh->size[d]);
    ADL_REQUIRE((mesh->link[d] & ~(0x3f01 | (d == 0 ? AUTODDL_FOLD : 0))) == 0,
                "mesh.link[%d] = %d: bit 0 = link class, bits 8..13 = allowed rows, bit 14 of link[0] = folded space", d, mesh->link[d]);
  }
  int64_t prod = 1;
  for (int d = 0; d < mesh->ndim; ++d) prod *= mesh->size[d];
  ADL_REQUIRE(prod <= (1 << 20), "mesh has %lld devices, at most 2^20 supported", (long long)prod);
  const int K = mesh_num_sigs(mesh);
  ADL_REQUIRE(K <= 256, "mesh.ndim = %d with %d signatures per layer: more than three levels need K <= 256 "
              "(restrict the rows per level, bits 8..13 of mesh.link)", mesh->ndim, K);
  if (out) {
    memset(out, 0, sizeof(*out));
    out->ndim = mesh->ndim;
    out->K = K;
    out->fold = fold ? 1 : 0;
    if (fold) out->ngroups = fold_groups(mesh, out->gfirst, out->glen);
    for (int d = 0; d < mesh->ndim; ++d) {
      out->size[d] = mesh->size[d];
      out->allow[d] = fold ? 0x07 : (((mesh->link[d] >> 8) & 0x3f) ? ((mesh->link[d] >> 8) & 0x3f) : 0x3f);
      out->magic_size[d] = (uint64_t)((((unsigned __int128)1 << 64) + mesh->size[d] - 1) / mesh->size[d]);
    }
    for (int m = 0; m < (1 << kTabLevels); ++m) {
      int64_t f = 1;
      for (int d = 0; d < mesh->ndim && d < kTabLevels; ++d)
        if (m >> d & 1) f *= mesh->size[d];
      out->sub[m] = (int32_t)f;
      out->magic_sub[m] = (uint64_t)((((unsigned __int128)1 << 64) + f - 1) / f);
    }
  }
  if (net) {
    for (int c = 0; c < 2; ++c) {
      ADL_REQUIRE(net->alpha_ps[c] >= 0 && net->alpha_ps[c] < ((int64_t)1 << 40), "net.alpha_ps[%d] out of range", c);
      ADL_REQUIRE(net->beta_ps_per_byte[c] >= 0 && net->beta_ps_per_byte[c] < ((int64_t)1 << 20),
                  "net.beta_ps_per_byte[%d] out of range", c);
    }
    ADL_REQUIRE(net->mem_cap_bytes >= 0, "net.mem_cap_bytes < 0");
    ADL_REQUIRE(net->micro_batches >= 0 && net->micro_batches < (1 << 20), "net.micro_batches out of range");
    if (out) {
      for (int d = 0; d < mesh->ndim; ++d) {
        out->alpha[d] = net->alpha_ps[mesh->link[d] & 1];
        out->beta[d] = net->beta_ps_per_byte[mesh->link[d] & 1];
      }
      out->mem_cap = net->mem_cap_bytes;
      out->accum = net->micro_batches > 1 ? net->micro_batches : 1;
    }
  }
  return AUTODDL_OK;
}

// valid ndim assumed (1..kMaxLevels).  R26: beyond three levels the index runs over the allowed rows only
int mesh_num_sigs(const autoddl_mesh* mesh) {
  if (mesh_folded(mesh)) {                                 // R28: ordered factorisations per group of equal levels
    int32_t first[kMaxLevels], len[kMaxLevels];
    const int ng = fold_groups(mesh, first, len);
    int64_t k = 1;
    for (int g = 0; g < ng; ++g) k *= (int64_t)(len[g] + 2) * (len[g] + 1) / 2;
    return k > (1 << 20) ? (1 << 20) : (int)k;
  }
  if (mesh->ndim <= 3) return mesh->ndim == 1 ? 6 : mesh->ndim == 2 ? 36 : 216;
  int64_t k = 1;
  for (int d = 0; d < mesh->ndim; ++d) {
    const int a = (mesh->link[d] >> 8) & 0x3f;
    k *= a ? __builtin_popcount(a) : 6;
  }
  return k > (1 << 20) ? (1 << 20) : (int)k;
}

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline size_t table_bytes(int64_t Bp, int64_t L, int64_t K) { return align_up((size_t)Bp * L * K * K * 8, 256); }
static inline bool bp_in_workspace(int64_t L, int64_t K) { return (size_t)L * K > 16 * 1024; }
static inline size_t bp_bytes(int64_t Bp, int64_t L, int64_t K) {
  return bp_in_workspace(L, K) ? align_up((size_t)Bp * L * K, 256) : 0;
}

// the fused build + DP kernel runs one chain per CTA: below this many chains the separate kernels (which spread the
// tiles of a chain over all SMs) are faster
static constexpr int32_t kFusedMinChains = 296;

// device-side address of a host pointer that lies in pinned, device-mapped memory (cudaHostAlloc / cudaHostRegister,
// e.g. a torch pin_memory() tensor); NULL for pageable memory
static const void* mapped_host_pointer(const void* h) {
  static const bool off = ADL_DEBUG_ENV("AUTODDL_NO_ZERO_COPY");
  if (off || !h) return nullptr;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, h) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  if (a.type != cudaMemoryTypeHost || a.devicePointer == nullptr) return nullptr;
  return a.devicePointer;
}

// Side stream of autoddl_search_host (per thread, per device): the optimum and its strategy are final when the chain DP
// is done, so their device-to-host copy runs beside the Coordinate Descent kernel instead of after it.
struct SideStream {
  int dev = -1;
  cudaStream_t stream = nullptr;
  cudaEvent_t dp_done = nullptr, copied = nullptr;
  bool ready() {
    static const bool off = ADL_DEBUG_ENV("AUTODDL_NO_D2H_OVERLAP");
    if (off) return false;
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); return false; }
    if (cur == dev && stream) return true;
    if (stream) { cudaStreamDestroy(stream); cudaEventDestroy(dp_done); cudaEventDestroy(copied); stream = nullptr; }
    if (cudaStreamCreateWithFlags(&stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&dp_done, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&copied, cudaEventDisableTiming) != cudaSuccess) {
      cudaGetLastError();
      stream = nullptr;
      return false;
    }
    dev = cur;
    return true;
  }
};
static thread_local SideStream g_side;

// Fork / join for the few-chain paths of autoddl_search: kernels that do not depend on one another (the K x K tables a
// caller wants, the chain DP, Coordinate Descent by look-ups) run side by side -- each of them fills only part of the
// machine.  Two side streams and their events per host thread and device; everything is ordered by events against the
// caller's stream: fork() after the last common producer, on(i) to launch on side stream i, join() before returning.
struct ForkStreams {
  int dev = -1;
  cudaStream_t s[2] = {nullptr, nullptr};
  cudaEvent_t forked = nullptr, done[2] = {nullptr, nullptr};
  bool used[2] = {false, false};
  bool ready() {
    static const bool off = ADL_DEBUG_ENV("AUTODDL_NO_FORK");
    if (off) return false;
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); return false; }
    if (cur == dev && s[0]) return true;
    if (s[0]) {
      for (int i = 0; i < 2; ++i) { cudaStreamDestroy(s[i]); cudaEventDestroy(done[i]); }
      cudaEventDestroy(forked);
      s[0] = nullptr;
    }
    bool ok = cudaEventCreateWithFlags(&forked, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i)
      ok = cudaStreamCreateWithFlags(&s[i], cudaStreamNonBlocking) == cudaSuccess &&
           cudaEventCreateWithFlags(&done[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { cudaGetLastError(); s[0] = nullptr; return false; }
    dev = cur;
    return true;
  }
  int fork(cudaStream_t main) {                            // what was launched on `main` so far precedes the side streams
    used[0] = used[1] = false;
    ADL_CUDA_CHECK(cudaEventRecord(forked, main));
    return AUTODDL_OK;
  }
  int on(int i, cudaStream_t* out) {
    if (!used[i]) { ADL_CUDA_CHECK(cudaStreamWaitEvent(s[i], forked, 0)); used[i] = true; }
    *out = s[i];
    return AUTODDL_OK;
  }
  int join(cudaStream_t main) {                            // `main` continues after the side streams' work
    for (int i = 0; i < 2; ++i)
      if (used[i]) {
        ADL_CUDA_CHECK(cudaEventRecord(done[i], s[i]));
        ADL_CUDA_CHECK(cudaStreamWaitEvent(main, done[i], 0));
        used[i] = false;
      }
    return AUTODDL_OK;
  }
};
static thread_local ForkStreams g_fork;

int device_sm_count() {
  int dev = 0, sms = 148;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    cudaGetLastError();
    sms = 148;
  }
  return sms;
}

static int check_device() {
  int n = 0;
  cudaError_t e = cudaGetDeviceCount(&n);
  if (e != cudaSuccess || n < 1) {
    set_error("no CUDA device available (%s); this library has no CPU fallback", cudaGetErrorString(e));
    cudaGetLastError();
    return AUTODDL_ECUDA;
  }
  return AUTODDL_OK;
}

}  // namespace autoddl

using namespace autoddl;

extern "C" {

int autoddl_num_signatures(const autoddl_mesh* mesh) {
  clear_error();
  int rc = validate_mesh_net(mesh, nullptr, nullptr);
  if (rc) return rc;
  return mesh_num_sigs(mesh);
}

size_t autoddl_workspace_bytes(int32_t Bp, int32_t L, int32_t S, const autoddl_mesh* mesh) {
  clear_error();
  MeshParams mp;
  if (validate_mesh_net(mesh, nullptr, &mp) || Bp < 1 || L < 1 || S < 0) return 0;
  const int64_t K = mesh_num_sigs(mesh);
  size_t b = table_bytes(Bp, L, K) + bp_bytes(Bp, L, K);
  const bool scan = chain_dp_scan_supported(mp, Bp, L);
  if (scan || cd_lookup_supported(mp, L, S)) b += factors_bytes(mp, Bp, L) + 256;
  if (scan) b += chain_dp_scan_bytes(mp, Bp, L);           // few long chains: the DP in class space, parallel over the layers
  if (chain_dp_scan_tab_supported((int32_t)K, Bp, L)) b += chain_dp_scan_tab_bytes((int32_t)K, Bp, L);   // the same on small tables
  if (cd_lookup_tab_supported((int32_t)K, L, S)) b += cd_lookup_tab_workspace_bytes((int32_t)K, Bp, L);   // best responses from small tables
  if (cd_lookup_supported(mp, L, S)) b += cd_lookup_workspace_bytes(mp, Bp, L) + 256;   // many starts: best responses
  if (mesh->ndim == 2) b += fused_bp_bytes(L) + align_up((size_t)Bp * S * L * 4, 256) + 256;   // fused kernel: back-pointers, strategies after sweep 1
  // autoddl_search_host staging: layers, init, opt_cost, strategy, cd_cost, cd_strategy, cd_sweeps
  b += align_up((size_t)Bp * L * sizeof(autoddl_layer), 256);
  b += align_up((size_t)Bp * S * L * 4, 256) * 2;
  b += align_up((size_t)Bp * 8, 256) + align_up((size_t)Bp * L * 4, 256);
  b += align_up((size_t)Bp * S * 8, 256) + align_up((size_t)Bp * S * 4, 256);
  return b;
}

int autoddl_build_tables(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const autoddl_mesh* mesh,
                         const autoddl_net* net, int64_t* d_T, int64_t* d_node, uint8_t* d_mask, void* stream) {
  clear_error();
  MeshParams mp;
  ADL_REQUIRE(net != nullptr, "net is NULL");
  int rc = validate_mesh_net(mesh, net, &mp);
  if (rc) return rc;
  ADL_REQUIRE(d_layers != nullptr && d_T != nullptr, "d_layers / d_T is NULL");
  ADL_REQUIRE(Bp >= 1 && L >= 1, "Bp = %d, L = %d must be >= 1", Bp, L);
  ADL_REQUIRE(((uintptr_t)d_T & 15) == 0, "d_T must be 16-byte aligned");
  ADL_REQUIRE(((uintptr_t)d_layers & 7) == 0 && ((uintptr_t)d_node & 7) == 0, "misaligned pointer");
  if ((rc = check_device())) return rc;
  return launch_build_tables(d_layers, Bp, L, mp, d_T, d_node, d_mask, (cudaStream_t)stream);
}

int autoddl_chain_dp(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const autoddl_mesh* mesh,
                     const autoddl_net* net, const int64_t* d_T, void* d_work, size_t work_bytes,
                     int64_t* d_opt_cost, int32_t* d_strategy, void* stream) {
  clear_error();
  MeshParams mp;
  int rc = validate_mesh_net(mesh, d_T ? nullptr : net, &mp);
  if (rc) return rc;
  ADL_REQUIRE(Bp >= 1 && L >= 1, "Bp = %d, L = %d must be >= 1", Bp, L);
  ADL_REQUIRE(d_opt_cost != nullptr && d_strategy != nullptr, "output pointer is NULL");
  ADL_REQUIRE(((uintptr_t)d_T & 15) == 0 && ((uintptr_t)d_work & 255) == 0, "d_T must be 16-byte, d_work 256-byte aligned");
  ADL_REQUIRE(((uintptr_t)d_opt_cost & 7) == 0 && ((uintptr_t)d_strategy & 3) == 0, "misaligned output pointer");
  if (!d_T) ADL_REQUIRE(d_layers != nullptr && net != nullptr, "d_T is NULL and no layers / net given");
  const int K = mp.K;
  cudaStream_t st = (cudaStream_t)stream;
  // many chains: the fused kernel (one chain per CTA, tables never leave shared memory); few chains: the fused kernel
  // would serialise the tiles of a chain on one CTA, so the tables are built by all SMs first when d_work can hold them
  if (!d_T && fused_build_dp_supported(mp, L) &&
      (Bp >= kFusedMinChains || d_work == nullptr || work_bytes < table_bytes(Bp, L, K) + bp_bytes(Bp, L, K))) {
    if (d_work == nullptr || work_bytes < fused_bp_bytes(L)) {
      set_error("chain_dp: workspace of %zu bytes needed, %zu given", fused_bp_bytes(L), d_work ? work_bytes : (size_t)0);
      return AUTODDL_EWORK;
    }
    if ((rc = check_device())) return rc;
    return launch_build_dp_fused(d_layers, Bp, L, mp, nullptr, nullptr, nullptr, d_opt_cost, d_strategy, (uint8_t*)d_work,
                                 nullptr, 0, nullptr, nullptr, st);
  }
  if (!d_T && chain_dp_scan_supported(mp, Bp, L)) {
    // few long chains, no table wanted: the factors (2.6 / 35.6 KB per layer) and the DP in class space on them
    const size_t fbytes = factors_bytes(mp, Bp, L);
    if (d_work != nullptr && work_bytes >= fbytes + chain_dp_scan_bytes(mp, Bp, L)) {
      if ((rc = check_device())) return rc;
      if ((rc = launch_build_factors(d_layers, Bp, L, mp, (int64_t*)d_work, st))) return rc;
      return launch_chain_dp_scan((const int64_t*)d_work, Bp, L, mp, (unsigned char*)d_work + fbytes, d_opt_cost, d_strategy, st);
    }
  }
  const size_t tb = d_T ? 0 : table_bytes(Bp, L, K), bb = bp_bytes(Bp, L, K);
  if (tb + bb > 0 && (d_work == nullptr || work_bytes < tb + bb)) {
    set_error("chain_dp: workspace of %zu bytes needed, %zu given", tb + bb, d_work ? work_bytes : (size_t)0);
    return AUTODDL_EWORK;
  }
  if ((rc = check_device())) return rc;
  if (!d_T) {
    if ((rc = launch_build_tables(d_layers, Bp, L, mp, (int64_t*)d_work, nullptr, nullptr, st))) return rc;
    d_T = (const int64_t*)d_work;
  }
  // few long chains on small tables (K <= 64): chunk products, prefix vectors, per-chunk DP -- parallel over the layers
  if (chain_dp_scan_tab_supported(K, Bp, L) && d_work != nullptr && work_bytes >= tb + chain_dp_scan_tab_bytes(K, Bp, L))
    return launch_chain_dp_scan_tab(d_T, Bp, L, K, (unsigned char*)d_work + tb, d_opt_cost, d_strategy, st);
  uint8_t* d_bp = bb ? (uint8_t*)d_work + tb : nullptr;
  return launch_chain_dp(d_T, Bp, L, K, d_bp, d_opt_cost, d_strategy, st);
}

int autoddl_coord_descent(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const autoddl_mesh* mesh,
                          const autoddl_net* net, const int64_t* d_T, void* d_work, size_t work_bytes,
                          const int32_t* d_init, int32_t S, int32_t max_sweeps, int64_t* d_cost,
                          int32_t* d_strategy, int32_t* d_sweeps, void* stream) {
  clear_error();
  MeshParams mp;
  int rc = validate_mesh_net(mesh, d_T ? nullptr : net, &mp);
  if (rc) return rc;
  ADL_REQUIRE(Bp >= 1 && L >= 1 && S >= 1 && max_sweeps >= 1, "Bp, L, S, max_sweeps must be >= 1");
  ADL_REQUIRE(d_init && d_cost && d_strategy && d_sweeps, "NULL pointer");
  ADL_REQUIRE(((uintptr_t)d_T & 15) == 0 && ((uintptr_t)d_work & 255) == 0, "d_T must be 16-byte, d_work 256-byte aligned");
  ADL_REQUIRE(((uintptr_t)d_cost & 7) == 0 && ((uintptr_t)d_strategy & 3) == 0 && ((uintptr_t)d_init & 3) == 0 &&
                  ((uintptr_t)d_sweeps & 3) == 0, "misaligned pointer");
  const int K = mp.K;
  cudaStream_t st = (cudaStream_t)stream;
  if (!d_T && cd_lookup_supported(mp, L, S)) {
    // many starts on library-built tables: no K x K table at all (factors -> best responses -> look-up sweeps)
    ADL_REQUIRE(d_layers != nullptr && net != nullptr, "d_T is NULL and no layers / net given");
    const size_t fbytes = factors_bytes(mp, Bp, L), need = fbytes + cd_lookup_workspace_bytes(mp, Bp, L);
    if (d_work == nullptr || work_bytes < need) {
      set_error("coord_descent: workspace of %zu bytes needed, %zu given", need, d_work ? work_bytes : (size_t)0);
      return AUTODDL_EWORK;
    }
    if ((rc = check_device())) return rc;
    if ((rc = launch_build_factors(d_layers, Bp, L, mp, (int64_t*)d_work, st))) return rc;
    return launch_cd_lookup((const int64_t*)d_work, Bp, L, mp, (unsigned char*)d_work + fbytes, d_init, S, max_sweeps, d_cost,
                            d_strategy, d_sweeps, st);
  }
  const size_t tb = d_T ? 0 : table_bytes(Bp, L, K);
  if (tb > 0 && (d_work == nullptr || work_bytes < tb)) {
    set_error("coord_descent: workspace of %zu bytes needed, %zu given", tb, d_work ? work_bytes : (size_t)0);
    return AUTODDL_EWORK;
  }
  if ((rc = check_device())) return rc;
  const bool built_here = d_T == nullptr && mp.ndim <= 3 && !mp.fold;  // tables of this library's builder (base-6 index): identical rows per class
  if (!d_T) {
    ADL_REQUIRE(d_layers != nullptr && net != nullptr, "d_T is NULL and no layers / net given");
    if ((rc = launch_build_tables(d_layers, Bp, L, mp, (int64_t*)d_work, nullptr, nullptr, st))) return rc;
    d_T = (const int64_t*)d_work;
  }
  // many starts on small tables (K <= 64): best responses from the tiles, then look-up sweeps
  if (cd_lookup_tab_supported(K, L, S) && d_work != nullptr && work_bytes >= tb + cd_lookup_tab_workspace_bytes(K, Bp, L))
    return launch_cd_lookup_tab(d_T, Bp, L, K, (unsigned char*)d_work + tb, d_init, S, max_sweeps, d_cost, d_strategy, d_sweeps, st);
  return launch_coord_descent(d_T, Bp, L, K, d_init, S, max_sweeps, d_cost, d_strategy, d_sweeps, st, false, built_here);
}

// (a1) -> (a2) -> (a3) on device pointers; tables go to d_T, or into d_work when d_T is NULL
static int search_device(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const MeshParams& mp, int K,
                         int64_t* d_T, int64_t* d_node, uint8_t* d_mask, unsigned char* d_work, size_t work_bytes,
                         int64_t* d_opt_cost, int32_t* d_strategy, const int32_t* d_init, int32_t S, int32_t max_sweeps,
                         int64_t* d_cd_cost, int32_t* d_cd_strategy, int32_t* d_cd_sweeps, cudaStream_t st) {
  const bool do_cd = d_init != nullptr;
  static const bool no_fuse = ADL_DEBUG_ENV("AUTODDL_NO_FUSE");         // debug builds only: three separate kernels
  const bool fused = !no_fuse && Bp >= kFusedMinChains && fused_build_dp_supported(mp, L);
  int rc;
  if (fused) {
    // ---- many chains on a two-level mesh: ONE kernel for tables + DP + the first two CD sweeps -----------------------------
    size_t used = 0;
    if (!d_T && do_cd) {                                    // the CD kernel that resumes reads the tables: keep them in d_work
      used = table_bytes(Bp, L, K);
      if (d_work == nullptr || work_bytes < used) {
        set_error("search: workspace of %zu bytes needed for the tables, %zu given", used, d_work ? work_bytes : (size_t)0);
        return AUTODDL_EWORK;
      }
      d_T = (int64_t*)d_work;
    }
    if (d_work == nullptr || work_bytes < used + fused_bp_bytes(L)) {
      set_error("search: workspace of %zu bytes needed, %zu given", used + fused_bp_bytes(L), d_work ? work_bytes : (size_t)0);
      return AUTODDL_EWORK;
    }
    // the first two CD sweeps ride in the fused kernel (the tile factors are in shared memory there); the CD kernel resumes
    // at sweep 3.  The strategies after sweep 1 go to a workspace slice behind the back-pointers.
    static const bool no_cd_fuse = ADL_DEBUG_ENV("AUTODDL_NO_CD_FUSE");
    const bool cd_resume = do_cd && !no_cd_fuse && fused_cd_sweep_supported(L, S);
    int32_t* d_cd_prev = nullptr;                           // strategies after sweep 1 when two sweeps were fused
    const size_t s1_off = (used + fused_bp_bytes(L) + 255) / 256 * 256;
    if (cd_resume && work_bytes >= s1_off + (size_t)Bp * S * L * 4) d_cd_prev = (int32_t*)(d_work + s1_off);
    if ((rc = launch_build_dp_fused(d_layers, Bp, L, mp, d_T, d_node, d_mask, d_opt_cost, d_strategy, d_work + used,
                                    cd_resume ? d_init : nullptr, S, cd_resume ? (d_cd_prev ? d_cd_prev : d_cd_strategy) : nullptr,
                                    cd_resume && d_cd_prev ? d_cd_strategy : nullptr, st)))
      return rc;
    if (g_mark) { cudaEventRecord(g_mark, st); g_mark = nullptr; }   // profiling hook: tables + DP done, CD kernel not yet started
    if (g_dp_done) { cudaEventRecord(g_dp_done, st); g_dp_done = nullptr; }
    if (!do_cd) return AUTODDL_OK;
    if (!cd_resume && cd_lookup_supported(mp, L, S)) {      // many starts per chain: best-response look-ups on the factors
      const size_t off = s1_off, fbytes = factors_bytes(mp, Bp, L);
      if (work_bytes >= off + fbytes + cd_lookup_workspace_bytes(mp, Bp, L)) {
        if ((rc = launch_build_factors(d_layers, Bp, L, mp, (int64_t*)(d_work + off), st))) return rc;
        return launch_cd_lookup((const int64_t*)(d_work + off), Bp, L, mp, d_work + off + fbytes, d_init, S, max_sweeps, d_cd_cost,
                                d_cd_strategy, d_cd_sweeps, st);
      }
    }
    return launch_coord_descent(d_T, Bp, L, K, d_init, S, max_sweeps, d_cd_cost, d_cd_strategy, d_cd_sweeps, st, cd_resume, true, d_cd_prev);
  }

  // ---- few chains, or another mesh: separate kernels.  Few long chains on two / three mesh levels take the DP in class space
  // on the factors (parallel over the layers); CD from >= 32 starts runs on the factors and their best-response tables.  A
  // K x K table is built only when the caller wants it (d_T, d_node, d_mask) or a kernel that reads it runs.
  const bool lookup = do_cd && cd_lookup_supported(mp, L, S);
  {
    const bool want_T = d_T != nullptr || d_node != nullptr || d_mask != nullptr || (do_cd && !lookup);
    const size_t tb = want_T && !d_T ? table_bytes(Bp, L, K) : 0, fbytes = factors_bytes(mp, Bp, L);
    const size_t sb = chain_dp_scan_supported(mp, Bp, L) ? chain_dp_scan_bytes(mp, Bp, L) : 0;
    const size_t brb = lookup ? cd_lookup_workspace_bytes(mp, Bp, L) : 0;
    if (sb && d_work != nullptr && work_bytes >= tb + fbytes + sb + brb) {
      int64_t* d_F = (int64_t*)(d_work + tb);
      if (want_T && !d_T) d_T = (int64_t*)d_work;
      // factors first; then the tables (if wanted), the DP on the factors and the look-up CD are independent of one another
      if ((rc = launch_build_factors(d_layers, Bp, L, mp, d_F, st))) return rc;
      const bool fork = (want_T || lookup) && g_fork.ready();
      cudaStream_t st_tab = st, st_cd = st;
      if (fork) {
        if ((rc = g_fork.fork(st))) return rc;
        if (want_T && (rc = g_fork.on(0, &st_tab))) return rc;
        if (lookup && (rc = g_fork.on(1, &st_cd))) return rc;
      }
      if (want_T && (rc = launch_build_tables(d_layers, Bp, L, mp, d_T, d_node, d_mask, st_tab))) return rc;
      if (lookup && (rc = launch_cd_lookup(d_F, Bp, L, mp, d_work + tb + fbytes + sb, d_init, S, max_sweeps, d_cd_cost, d_cd_strategy,
                                           d_cd_sweeps, st_cd)))
        return rc;
      if ((rc = launch_chain_dp_scan(d_F, Bp, L, mp, d_work + tb + fbytes, d_opt_cost, d_strategy, st))) return rc;
      if (g_mark) { cudaEventRecord(g_mark, st); g_mark = nullptr; }
      if (g_dp_done) { cudaEventRecord(g_dp_done, st); g_dp_done = nullptr; }
      if (fork && (rc = g_fork.join(st))) return rc;
      if (!do_cd || lookup) return AUTODDL_OK;
      return launch_coord_descent(d_T, Bp, L, K, d_init, S, max_sweeps, d_cd_cost, d_cd_strategy, d_cd_sweeps, st, false, true);
    }
  }
  const size_t tb = d_T ? 0 : table_bytes(Bp, L, K), bb = bp_bytes(Bp, L, K);
  if (tb + bb > 0 && (d_work == nullptr || work_bytes < tb + bb)) {
    set_error("search: workspace of %zu bytes needed, %zu given", tb + bb, d_work ? work_bytes : (size_t)0);
    return AUTODDL_EWORK;
  }
  if (!d_T) d_T = (int64_t*)d_work;
  if ((rc = launch_build_tables(d_layers, Bp, L, mp, d_T, d_node, d_mask, st))) return rc;
  const bool scan_tab = chain_dp_scan_tab_supported((int32_t)K, Bp, L) && work_bytes >= tb + chain_dp_scan_tab_bytes((int32_t)K, Bp, L);
  // small tables, few long chains, many starts: the layer-parallel DP and the look-up CD both read the tables and nothing
  // else -- side by side, each with its own slice of the workspace
  const size_t stb = scan_tab ? align_up(chain_dp_scan_tab_bytes((int32_t)K, Bp, L), 256) : 0;
  const bool cd_beside = scan_tab && do_cd && !lookup && cd_lookup_tab_supported((int32_t)K, L, S) &&
                         work_bytes >= tb + stb + cd_lookup_tab_workspace_bytes((int32_t)K, Bp, L) && g_fork.ready();
  if (cd_beside) {
    cudaStream_t st_cd = st;
    if ((rc = g_fork.fork(st)) || (rc = g_fork.on(1, &st_cd))) return rc;
    if ((rc = launch_cd_lookup_tab(d_T, Bp, L, (int32_t)K, d_work + tb + stb, d_init, S, max_sweeps, d_cd_cost, d_cd_strategy, d_cd_sweeps, st_cd)))
      return rc;
  }
  // few chains on larger tables: the DP (a cluster or a CTA per chain) and the gather CD (a warp per start) fill a fraction
  // of the machine each and read the tables only (the gather kernel needs no workspace)
  const bool gather_beside = !cd_beside && do_cd && !lookup && Bp <= 64 && !cd_lookup_tab_supported((int32_t)K, L, S) && g_fork.ready();
  if (gather_beside) {
    cudaStream_t st_cd = st;
    if ((rc = g_fork.fork(st)) || (rc = g_fork.on(1, &st_cd))) return rc;
    if ((rc = launch_coord_descent(d_T, Bp, L, K, d_init, S, max_sweeps, d_cd_cost, d_cd_strategy, d_cd_sweeps, st_cd, false,
                                   mp.ndim <= 3 && !mp.fold)))
      return rc;
  }
  if (scan_tab) rc = launch_chain_dp_scan_tab(d_T, Bp, L, (int32_t)K, d_work + tb, d_opt_cost, d_strategy, st);
  else rc = launch_chain_dp(d_T, Bp, L, K, bb ? d_work + tb : nullptr, d_opt_cost, d_strategy, st);
  if (rc) return rc;
  if (g_mark) { cudaEventRecord(g_mark, st); g_mark = nullptr; }
  if (g_dp_done) { cudaEventRecord(g_dp_done, st); g_dp_done = nullptr; }
  if (cd_beside || gather_beside) return g_fork.join(st);
  if (!do_cd) return AUTODDL_OK;
  if (lookup) {
    const size_t off = align_up(tb + bb, 256), fbytes = factors_bytes(mp, Bp, L);
    if (work_bytes >= off + fbytes + cd_lookup_workspace_bytes(mp, Bp, L)) {
      if ((rc = launch_build_factors(d_layers, Bp, L, mp, (int64_t*)(d_work + off), st))) return rc;
      return launch_cd_lookup((const int64_t*)(d_work + off), Bp, L, mp, d_work + off + fbytes, d_init, S, max_sweeps, d_cd_cost,
                              d_cd_strategy, d_cd_sweeps, st);
    }
  }
  if (cd_lookup_tab_supported((int32_t)K, L, S) && work_bytes >= tb + cd_lookup_tab_workspace_bytes((int32_t)K, Bp, L))
    return launch_cd_lookup_tab(d_T, Bp, L, (int32_t)K, d_work + tb, d_init, S, max_sweeps, d_cd_cost, d_cd_strategy, d_cd_sweeps, st);
  return launch_coord_descent(d_T, Bp, L, K, d_init, S, max_sweeps, d_cd_cost, d_cd_strategy, d_cd_sweeps, st, false, mp.ndim <= 3 && !mp.fold);
}

int autoddl_search(const autoddl_layer* d_layers, int32_t Bp, int32_t L, const autoddl_mesh* mesh, const autoddl_net* net,
                   int64_t* d_T, int64_t* d_node, uint8_t* d_mask, void* d_work, size_t work_bytes, int64_t* d_opt_cost,
                   int32_t* d_strategy, const int32_t* d_init, int32_t S, int32_t max_sweeps, int64_t* d_cd_cost,
                   int32_t* d_cd_strategy, int32_t* d_cd_sweeps, void* stream) {
  clear_error();
  MeshParams mp;
  ADL_REQUIRE(net != nullptr, "net is NULL");
  int rc = validate_mesh_net(mesh, net, &mp);
  if (rc) return rc;
  ADL_REQUIRE(d_layers != nullptr && d_opt_cost != nullptr && d_strategy != nullptr, "NULL pointer");
  ADL_REQUIRE(Bp >= 1 && L >= 1, "Bp = %d, L = %d must be >= 1", Bp, L);
  if (d_init) {
    ADL_REQUIRE(S >= 1 && max_sweeps >= 1, "S, max_sweeps must be >= 1");
    ADL_REQUIRE(d_cd_cost && d_cd_strategy && d_cd_sweeps, "NULL Coordinate Descent output");
  }
  ADL_REQUIRE(((uintptr_t)d_T & 15) == 0 && ((uintptr_t)d_work & 255) == 0, "d_T must be 16-byte, d_work 256-byte aligned");
  ADL_REQUIRE(((uintptr_t)d_layers & 7) == 0 && ((uintptr_t)d_node & 7) == 0 && ((uintptr_t)d_opt_cost & 7) == 0 &&
                  ((uintptr_t)d_cd_cost & 7) == 0 && ((uintptr_t)d_strategy & 3) == 0 && ((uintptr_t)d_init & 3) == 0 &&
                  ((uintptr_t)d_cd_strategy & 3) == 0 && ((uintptr_t)d_cd_sweeps & 3) == 0, "misaligned pointer");
  if ((rc = check_device())) return rc;
  return search_device(d_layers, Bp, L, mp, mp.K, d_T, d_node, d_mask, (unsigned char*)d_work, work_bytes,
                       d_opt_cost, d_strategy, d_init, S, max_sweeps, d_cd_cost, d_cd_strategy, d_cd_sweeps, (cudaStream_t)stream);
}

int autoddl_search_host(const autoddl_layer* h_layers, int32_t Bp, int32_t L, const autoddl_mesh* mesh,
                        const autoddl_net* net, const int32_t* h_init, int32_t S, int32_t max_sweeps,
                        void* d_work, size_t work_bytes, int64_t* h_opt_cost, int32_t* h_strategy,
                        int64_t* h_cd_cost, int32_t* h_cd_strategy, int32_t* h_cd_sweeps, void* stream) {
  clear_error();
  MeshParams mp;
  ADL_REQUIRE(net != nullptr, "net is NULL");
  int rc = validate_mesh_net(mesh, net, &mp);
  if (rc) return rc;
  ADL_REQUIRE(h_layers != nullptr, "h_layers is NULL");
  ADL_REQUIRE(Bp >= 1 && L >= 1, "Bp = %d, L = %d must be >= 1", Bp, L);
  const bool do_cd = h_init != nullptr;
  if (do_cd) ADL_REQUIRE(S >= 1 && max_sweeps >= 1, "S, max_sweeps must be >= 1");
  if (!do_cd) S = 0;
  ADL_REQUIRE(((uintptr_t)d_work & 255) == 0, "d_work must be 256-byte aligned");
  const size_t need = autoddl_workspace_bytes(Bp, L, S, mesh);
  if (d_work == nullptr || work_bytes < need) {
    set_error("search_host: workspace of %zu bytes needed, %zu given", need, d_work ? work_bytes : (size_t)0);
    return AUTODDL_EWORK;
  }
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int K = mp.K;

  unsigned char* w = (unsigned char*)d_work;
  auto carve = [&](size_t bytes) { unsigned char* p = w; w += align_up(bytes, 256); return p; };
  size_t tables_region = table_bytes(Bp, L, K) + bp_bytes(Bp, L, K) +
                         (mesh->ndim == 2 ? fused_bp_bytes(L) + align_up((size_t)Bp * S * L * 4, 256) + 256 : 0);
  if (chain_dp_scan_supported(mp, Bp, L) || (do_cd && cd_lookup_supported(mp, L, S))) tables_region += factors_bytes(mp, Bp, L) + 256;
  if (chain_dp_scan_supported(mp, Bp, L)) tables_region += chain_dp_scan_bytes(mp, Bp, L);
  if (chain_dp_scan_tab_supported((int32_t)K, Bp, L)) tables_region += chain_dp_scan_tab_bytes((int32_t)K, Bp, L);
  if (do_cd && cd_lookup_tab_supported((int32_t)K, L, S)) tables_region += cd_lookup_tab_workspace_bytes((int32_t)K, Bp, L);
  if (do_cd && cd_lookup_supported(mp, L, S)) tables_region += cd_lookup_workspace_bytes(mp, Bp, L) + 512;
  unsigned char* d_tables = carve(tables_region);                                   // tables, then back-pointers
  autoddl_layer* d_layers = (autoddl_layer*)carve((size_t)Bp * L * sizeof(autoddl_layer));
  int32_t* d_init = (int32_t*)carve((size_t)Bp * S * L * 4);
  int32_t* d_cd_strategy = (int32_t*)carve((size_t)Bp * S * L * 4);
  int64_t* d_opt = (int64_t*)carve((size_t)Bp * 8);
  int32_t* d_strategy = (int32_t*)carve((size_t)Bp * L * 4);
  int64_t* d_cd_cost = (int64_t*)carve((size_t)Bp * S * 8);
  int32_t* d_cd_sweeps = (int32_t*)carve((size_t)Bp * S * 4);

  // Inputs in pinned (page-locked, device-mapped) host memory are read by the kernels straight over PCIe: every record
  // and every start is read once, the reads overlap the table stores, and the explicit copy (0.3 ms for config 4)
  // disappears.  Pageable inputs are copied first.
  const autoddl_layer* k_layers = (const autoddl_layer*)mapped_host_pointer(h_layers);
  if (!k_layers) {
    ADL_CUDA_CHECK(cudaMemcpyAsync(d_layers, h_layers, (size_t)Bp * L * sizeof(autoddl_layer), cudaMemcpyHostToDevice, st));
    k_layers = d_layers;
  }
  const int32_t* k_init = nullptr;
  if (do_cd) {
    k_init = (const int32_t*)mapped_host_pointer(h_init);
    if (!k_init) {
      ADL_CUDA_CHECK(cudaMemcpyAsync(d_init, h_init, (size_t)Bp * S * L * 4, cudaMemcpyHostToDevice, st));
      k_init = d_init;
    }
  }
  const bool overlap = do_cd && (h_opt_cost || h_strategy) && g_side.ready();
  if (overlap) g_dp_done = g_side.dp_done;
  rc = search_device(k_layers, Bp, L, mp, K, nullptr, nullptr, nullptr, d_tables, tables_region,
                     d_opt, d_strategy, k_init, S, max_sweeps, d_cd_cost, d_cd_strategy, d_cd_sweeps, st);
  const bool dp_recorded = overlap && g_dp_done == nullptr;
  g_dp_done = nullptr;
  if (rc) return rc;
  cudaStream_t dp_st = st;
  if (dp_recorded) {                                        // copy the DP results while Coordinate Descent runs
    ADL_CUDA_CHECK(cudaStreamWaitEvent(g_side.stream, g_side.dp_done, 0));
    dp_st = g_side.stream;
  }
  if (h_opt_cost) ADL_CUDA_CHECK(cudaMemcpyAsync(h_opt_cost, d_opt, (size_t)Bp * 8, cudaMemcpyDeviceToHost, dp_st));
  if (h_strategy) ADL_CUDA_CHECK(cudaMemcpyAsync(h_strategy, d_strategy, (size_t)Bp * L * 4, cudaMemcpyDeviceToHost, dp_st));
  if (dp_recorded) {
    ADL_CUDA_CHECK(cudaEventRecord(g_side.copied, g_side.stream));
    ADL_CUDA_CHECK(cudaStreamWaitEvent(st, g_side.copied, 0));          // the final synchronise covers both streams
  }
  if (do_cd) {
    if (h_cd_cost) ADL_CUDA_CHECK(cudaMemcpyAsync(h_cd_cost, d_cd_cost, (size_t)Bp * S * 8, cudaMemcpyDeviceToHost, st));
    if (h_cd_strategy)
      ADL_CUDA_CHECK(cudaMemcpyAsync(h_cd_strategy, d_cd_strategy, (size_t)Bp * S * L * 4, cudaMemcpyDeviceToHost, st));
    if (h_cd_sweeps) ADL_CUDA_CHECK(cudaMemcpyAsync(h_cd_sweeps, d_cd_sweeps, (size_t)Bp * S * 4, cudaMemcpyDeviceToHost, st));
  }
  ADL_CUDA_CHECK(cudaStreamSynchronize(st));
  return AUTODDL_OK;
}

int autoddl_metropolis(const int64_t* d_T, int32_t Bp, int32_t L, const autoddl_mesh* mesh, const int32_t* d_init,
                       int32_t S, int32_t nsteps, int64_t tau_ps, uint64_t seed, int64_t* d_best_cost,
                       int32_t* d_best_strategy, int64_t* d_final_cost, int32_t* d_final_strategy, int32_t* d_accepted,
                       void* stream) {
  clear_error();
  int rc = validate_mesh_net(mesh, nullptr, nullptr);
  if (rc) return rc;
  ADL_REQUIRE(Bp >= 1 && L >= 1 && S >= 1 && nsteps >= 0, "Bp, L, S must be >= 1 and nsteps >= 0");
  ADL_REQUIRE(tau_ps >= 0 && tau_ps < ((int64_t)1 << 40), "tau_ps must lie in [0, 2^40)");
  ADL_REQUIRE(d_T && d_init && d_best_cost && d_best_strategy && d_final_cost && d_final_strategy && d_accepted, "NULL pointer");
  ADL_REQUIRE(((uintptr_t)d_T & 7) == 0 && ((uintptr_t)d_best_cost & 7) == 0 && ((uintptr_t)d_final_cost & 7) == 0 &&
                  ((uintptr_t)d_init & 3) == 0 && ((uintptr_t)d_best_strategy & 3) == 0 &&
                  ((uintptr_t)d_final_strategy & 3) == 0 && ((uintptr_t)d_accepted & 3) == 0, "misaligned pointer");
  if ((rc = check_device())) return rc;
  return launch_metropolis(d_T, Bp, L, mesh_num_sigs(mesh), d_init, S, nsteps, tau_ps, seed, d_best_cost, d_best_strategy,
                           d_final_cost, d_final_strategy, d_accepted, (cudaStream_t)stream);
}

size_t autoddl_fit_workspace_bytes(void) { return fit_workspace_bytes(); }

int autoddl_fit_alpha_beta(const int32_t* d_kind, const int32_t* d_p, const int64_t* d_bytes, const double* d_time,
                           int64_t N, double* d_out, void* d_work, size_t work_bytes, void* stream) {
  clear_error();
  ADL_REQUIRE(d_kind && d_p && d_bytes && d_time && d_out, "NULL pointer");
  ADL_REQUIRE(N >= 1, "N must be >= 1");
  ADL_REQUIRE(((uintptr_t)d_bytes & 7) == 0 && ((uintptr_t)d_time & 7) == 0 && ((uintptr_t)d_out & 7) == 0 &&
                  ((uintptr_t)d_work & 7) == 0 && ((uintptr_t)d_kind & 3) == 0 && ((uintptr_t)d_p & 3) == 0, "misaligned pointer");
  if (d_work == nullptr || work_bytes < fit_workspace_bytes()) {
    set_error("fit_alpha_beta: workspace of %zu bytes needed, %zu given", fit_workspace_bytes(), d_work ? work_bytes : (size_t)0);
    return AUTODDL_EWORK;
  }
  int rc = check_device();
  if (rc) return rc;
  return launch_fit_alpha_beta(d_kind, d_p, d_bytes, d_time, N, d_out, (double*)d_work, (cudaStream_t)stream);
}

int autoddl_best_of_starts(const int64_t* d_cost, int32_t Bp, int32_t S, int64_t* d_best_cost, int32_t* d_best_start,
                           void* stream) {
  clear_error();
  ADL_REQUIRE(d_cost && d_best_cost && d_best_start, "NULL pointer");
  ADL_REQUIRE(Bp >= 1 && S >= 1, "Bp, S must be >= 1");
  ADL_REQUIRE(((uintptr_t)d_cost & 7) == 0 && ((uintptr_t)d_best_cost & 7) == 0 && ((uintptr_t)d_best_start & 3) == 0, "misaligned pointer");
  int rc = check_device();
  if (rc) return rc;
  return launch_best_of_starts(d_cost, Bp, S, d_best_cost, d_best_start, (cudaStream_t)stream);
}

size_t autoddl_pipeline_workspace_bytes(int32_t L, int32_t K, int32_t stages) {
  if (L < 1 || K < 1 || stages < 1) return 0;
  const size_t a = partition_workspace_bytes(L, stages), b = align_up((size_t)L * K, 256) + 256;
  return a > b ? a : b;
}

int autoddl_segment_optima(const int64_t* d_T, const int64_t* d_node, const uint8_t* d_mask, int32_t L, const autoddl_mesh* mesh,
                           int64_t* d_tri, void* stream) {
  clear_error();
  int rc = validate_mesh_net(mesh, nullptr, nullptr);
  if (rc) return rc;
  ADL_REQUIRE(d_T && d_node && d_mask && d_tri, "NULL pointer");
  ADL_REQUIRE(L >= 1, "L must be >= 1");
  ADL_REQUIRE(((uintptr_t)d_T & 7) == 0 && ((uintptr_t)d_node & 7) == 0 && ((uintptr_t)d_tri & 7) == 0, "misaligned pointer");
  if ((rc = check_device())) return rc;
  return launch_segment_optima(d_T, d_node, d_mask, L, mesh_num_sigs(mesh), d_tri, (cudaStream_t)stream);
}

int autoddl_stage_transfer(const autoddl_layer* d_layers, int32_t L, const autoddl_mesh* mesh, const autoddl_net* net,
                           int64_t* d_xfer, void* stream) {
  clear_error();
  MeshParams mp;
  ADL_REQUIRE(net != nullptr, "net is NULL");
  int rc = validate_mesh_net(mesh, net, &mp);
  if (rc) return rc;
  ADL_REQUIRE(d_layers && d_xfer, "NULL pointer");
  ADL_REQUIRE(L >= 1, "L must be >= 1");
  ADL_REQUIRE(((uintptr_t)d_layers & 7) == 0 && ((uintptr_t)d_xfer & 7) == 0, "misaligned pointer");
  if ((rc = check_device())) return rc;
  int64_t q = 1;
  for (int d = 0; d < mesh->ndim; ++d) q *= mesh->size[d];
  return launch_stage_transfer(d_layers, L, q, mp.accum, net->alpha_ps[1], net->beta_ps_per_byte[1], d_xfer, (cudaStream_t)stream);
}

int autoddl_pipeline_partition(const int64_t* d_tri, const int64_t* d_xfer, int32_t L, int32_t stages, int32_t objective,
                               void* d_work, size_t work_bytes, int64_t* d_value, int32_t* d_cuts, void* stream) {
  clear_error();
  ADL_REQUIRE(d_tri && d_xfer && d_value && d_cuts, "NULL pointer");
  ADL_REQUIRE(L >= 1 && stages >= 1 && stages <= L, "need 1 <= stages <= L");
  ADL_REQUIRE(objective == 0 || objective == 1, "objective: 0 = sum of the stage costs, 1 = max");
  ADL_REQUIRE(((uintptr_t)d_tri & 7) == 0 && ((uintptr_t)d_xfer & 7) == 0 && ((uintptr_t)d_value & 7) == 0 &&
                  ((uintptr_t)d_cuts & 3) == 0 && ((uintptr_t)d_work & 255) == 0, "misaligned pointer");
  if (d_work == nullptr || work_bytes < partition_workspace_bytes(L, stages)) {
    set_error("pipeline_partition: workspace of %zu bytes needed, %zu given", partition_workspace_bytes(L, stages), d_work ? work_bytes : (size_t)0);
    return AUTODDL_EWORK;
  }
  int rc = check_device();
  if (rc) return rc;
  return launch_partition(d_tri, d_xfer, L, stages, objective, d_work, d_value, d_cuts, (cudaStream_t)stream);
}

int autoddl_segment_strategies(const int64_t* d_T, const int64_t* d_node, const uint8_t* d_mask, int32_t L,
                               const autoddl_mesh* mesh, const int32_t* d_cuts, int32_t stages, void* d_work, size_t work_bytes,
                               int64_t* d_seg_cost, int32_t* d_strategy, void* stream) {
  clear_error();
  int rc = validate_mesh_net(mesh, nullptr, nullptr);
  if (rc) return rc;
  ADL_REQUIRE(d_T && d_node && d_mask && d_cuts && d_seg_cost && d_strategy, "NULL pointer");
  ADL_REQUIRE(L >= 1 && stages >= 1 && stages <= L, "need 1 <= stages <= L");
  const int K = mesh_num_sigs(mesh);
  if (d_work == nullptr || work_bytes < (size_t)L * K) {
    set_error("segment_strategies: workspace of %zu bytes needed, %zu given", (size_t)L * K, d_work ? work_bytes : (size_t)0);
    return AUTODDL_EWORK;
  }
  if ((rc = check_device())) return rc;
  return launch_segment_strategies(d_T, d_node, d_mask, L, K, d_cuts, stages, (uint8_t*)d_work, d_seg_cost, d_strategy,
                                   (cudaStream_t)stream);
}

int autoddl_store_probe(int64_t* d_T, int32_t Bp, int32_t L, int32_t K, void* stream) {
  clear_error();
  ADL_REQUIRE(d_T != nullptr && Bp >= 1 && L >= 1 && K >= 1 && K <= 256 && (K * K) % 2 == 0, "store_probe: bad arguments");
  ADL_REQUIRE(((uintptr_t)d_T & 15) == 0, "store_probe: misaligned");
  int rc = check_device();
  if (rc) return rc;
  return launch_store_probe(d_T, Bp, L, K * K, (cudaStream_t)stream);
}

int autoddl_copy_probe(const void* d_src, void* d_dst, size_t bytes, void* stream) {
  clear_error();
  ADL_REQUIRE(d_src && d_dst && bytes > 0 && bytes % 16 == 0, "copy_probe: bad arguments");
  ADL_REQUIRE(((uintptr_t)d_src & 15) == 0 && ((uintptr_t)d_dst & 15) == 0, "copy_probe: misaligned");
  int rc = check_device();
  if (rc) return rc;
  return launch_copy_probe(d_src, d_dst, bytes, (cudaStream_t)stream);
}

int autoddl_profile_mark(void* cuda_event) {
  g_mark = (cudaEvent_t)cuda_event;
  return AUTODDL_OK;
}

int64_t autoddl_launch_count(void) { return g_launches; }

const char* autoddl_last_error(void) { return g_err; }

}  // extern "C"
