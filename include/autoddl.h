/*
 * include/autoddl.h -- C-ABI boundary of the B200-native AutoDDL strategy-search hot path.
 *
 * What it computes (citations are lines of the paper text PAPER.md, arxiv 2301.06813; the exact
 * readings R1..R25 are listed in DESIGN.md section 3):
 *   (a1) autoddl_build_tables   SBP cost tables: redistribution cost between every producer-output /
 *        consumer-input signature pair (collectives of Table 2 PAPER.md:102-108,
 *        intra/inter-node link rule PAPER.md:203) + weight-gradient all-reduce
 *        + per-device memory feasibility.
 *   (a2) autoddl_chain_dp       exact optimum over all K^L strategies of a chain (the result of the
 *        paper's "exhaustive search") by min-plus dynamic programming.
 *   (a3) autoddl_coord_descent  the paper's Coordinate Descent, many starts.
 *   (f2) autoddl_metropolis     the paper's Metropolis-Hastings sampler, many chains.
 *
 * Conventions
 *   - All costs are int64 picoseconds.  PEN = 2^50 is added to every cell whose consumer signature
 *     is infeasible; Cost < 2^50  <=>  strategy feasible.
 *   - d_* arguments are DEVICE pointers owned by the caller, h_* are HOST pointers.  `mesh` and
 *     `net` are host pointers, read before the call returns.  `stream` is a cudaStream_t (NULL =
 *     default stream).  Calls taking only d_* pointers are asynchronous on `stream`; they allocate
 *     nothing and never synchronise.  autoddl_search_host synchronises `stream` before returning.
 *   - Layouts are dense row-major:  T[Bp][L][K][K] (i = producer signature = row, j = consumer
 *     signature = column), node[Bp][L][K], mask[Bp][L][K], strategy[Bp][L], init[Bp][S][L],
 *     cd_strategy[Bp][S][L], cd_cost[Bp][S], cd_sweeps[Bp][S].   K = autoddl_num_signatures(mesh).
 *   - d_T must be 16-byte aligned; all other pointers naturally aligned.
 *   - Return value: 0 success, AUTODDL_EINVAL (-1) bad argument, AUTODDL_ECUDA (-2) CUDA runtime
 *     error, AUTODDL_EWORK (-3) workspace too small.  Text via autoddl_last_error() (thread-local).
 *     There is no CPU fallback: without a CUDA device every compute entry point returns ECUDA.
 */
#ifndef AUTODDL_H
#define AUTODDL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AUTODDL_OK      0
#define AUTODDL_EINVAL (-1)
#define AUTODDL_ECUDA  (-2)
#define AUTODDL_EWORK  (-3)

#define AUTODDL_PEN ((int64_t)1 << 50)

/* layer kinds */
#define AUTODDL_GEMM 0   /* O[M,N] = I[M,Kd] W[Kd,N] */
#define AUTODDL_ATTN 1   /* weightless; partial-sum signatures are invalid                 */

/* One layer of the chain, 64 bytes.  PAPER.md:189-193. */
typedef struct {
  int64_t M, Kd, N;          /* GEMM shape; ATTN: Kd = 0, N = hidden                                 */
  int64_t in_rows, in_cols;  /* the activation that is redistributed INTO this layer (consumer side) */
  int32_t kind;              /* AUTODDL_GEMM / AUTODDL_ATTN                                          */
  int32_t act_bytes;         /* bytes per activation (and activation-gradient) element               */
  int32_t wgrad_bytes;       /* bytes per weight-gradient element (the all-reduce message)           */
  int32_t wstate_bytes;      /* resident bytes per weight element (weight + grad + optimiser state)  */
  int32_t max_split_rows;    /* largest allowed total split of axis 0                 */
  int32_t max_split_cols;    /* largest allowed total split of the output's axis 1                   */
} autoddl_layer;

/* Device mesh, level 0 outermost.  link[d] bit 0: 0 = intra-node (NVLink), 1 = inter-node.
 * link[d] bits 8..13 (optional): the signature rows allowed on the level, bit g = row g of the per-level table
 * (0 split rows, 1 split columns, 2 split the reduction dim, 3 replicate, 4 partial input, 5 partial weight); 0 = all
 * six.  With 0x07 << 8 on every level of a mesh refined into prime sub-levels the feasible strategies are exactly the
 * paper's SBP matmul factorisations I = (S0:p0, B:p1, S1:p2), W = (B, S1, S0), O = (S0, S1, P);
 * disallowed signatures are infeasible (penalty 2^50, mask 0).  For ndim <= 3, K stays 6^ndim.
 * ndim = 4, 5 (R26; 2 nodes x 8 GPUs = 2 | 2.2.2, the paper's 2 x 16 GPUs = 2 | 2.2.2.2): the
 * signature index runs over the ALLOWED rows only, a mixed-radix number with level 0 most significant whose digit x
 * on level d names the x-th allowed row of that level in increasing order; K = product of the levels' allowed-row
 * counts and must be <= 256 (81 / 243 with 0x07 << 8 on every level). */
/* FOLDED factorisation space (R28): bit 14 (AUTODDL_FOLD) of link[0].  Rows {0,1,2} on every level (bits 8..13
 * are ignored), ndim up to 8, and inside every group of consecutive levels with equal size and link class only the
 * sorted digit strings 0..0 1..1 2..2 are signatures: one signature per ordered factorisation p = p0 p1 p2 of the group
 * -- with an inter-node group followed by an intra-node group these are the paper's (nodes, GPUs) tuples per SBP
 * dimension.  The index is a mixed-radix number over the groups, group 0 most significant; the digit
 * of a group of n levels enumerates its (n + 2)(n + 1) / 2 strings in increasing lexicographic order (p0 descending,
 * then p1 descending); K = the product over the groups, <= 256 (28 / 36 / 45 for 2^6 / 2^7 / 2^8 single-GPU nodes).
 * Costs are those of the same digit strings in the per-level encoding above. */
#define AUTODDL_MAX_LEVELS 8
#define AUTODDL_FOLD 0x4000
typedef struct { int32_t ndim; int32_t size[AUTODDL_MAX_LEVELS]; int32_t link[AUTODDL_MAX_LEVELS]; } autoddl_mesh;

/* alpha-beta parameters per link class; mem_cap_bytes 0 = no cap.
 * micro_batches: gradient accumulation: the activation redistributions of a cell are paid once per
 * micro-batch, the weight-gradient all-reduce once per mini-batch: T = m * edge + node + penalty; 0 or 1 = none.
 * Must be < 2^20.  48 bytes. */
typedef struct { int64_t alpha_ps[2]; int64_t beta_ps_per_byte[2]; int64_t mem_cap_bytes; int64_t micro_batches; } autoddl_net;

/* K = 6^ndim for ndim <= 3, the product of the allowed-row counts for ndim = 4, 5, the number of ordered factorisations
 * in the folded space; or AUTODDL_EINVAL. Host only. */
int autoddl_num_signatures(const autoddl_mesh* mesh);

/* Bytes of device workspace that any entry point below may need for (Bp, L, S): the tables when
 * d_T is NULL, DP back-pointers, and autoddl_search_host's staging.  Host only. */
size_t autoddl_workspace_bytes(int32_t Bp, int32_t L, int32_t S, const autoddl_mesh* mesh);

/* (a1) Build T, node, mask for Bp chains of L layers.  d_node / d_mask may be NULL.
 * Accepted ranges (checked, AUTODDL_EINVAL otherwise): 1 <= mesh.size[d] <= 65536 and at most 2^20 devices in all;
 * 0 <= alpha_ps < 2^40; 0 <= beta_ps_per_byte < 2^20; 0 <= micro_batches < 2^20; mem_cap_bytes >= 0.
 * Caller's obligation (NOT checked: the records live on the device): every extent of a layer record is >= 1 and the
 * products rows * cols * bytes * beta * micro_batches stay below 2^50, so that a cell is below 2^51 and no int64
 * product or sum overflows; real workloads (the paper's 2^20 x 8192 fp32 activations at 80 ps/B) are below 2^44. */
int autoddl_build_tables(const autoddl_layer* d_layers, int32_t Bp, int32_t L,
                         const autoddl_mesh* mesh, const autoddl_net* net,
                         int64_t* d_T, int64_t* d_node, uint8_t* d_mask, void* stream);

/* (a2) f_0[j] = T[0][0][j]; f_l[j] = min_i f_{l-1}[i] + T[l][i][j]; smallest index wins every tie;
 * backtrack from the smallest argmin of f_{L-1}.  d_T == NULL: the tables are computed from d_layers
 * -- on a 2-level mesh (K = 36), for >= 296 chains or when d_work cannot hold the tables, inside the DP kernel
 * itself (one warp per chain, every tile in factor form in shared memory, never stored); at most 64 chains of at least
 * 32 layers on a 2- or 3-level mesh are solved in class space, parallel over the layers, from the tiles' factors alone
 * (no K x K table is formed; same optimum, same tie-break); otherwise the tables are first built into
 * d_work.  d_work (>= autoddl_workspace_bytes) also holds back-pointers (fused kernel: only for chains too long for
 * shared memory; separate kernel: when L * K > 16384) and the class matrices of that path; with less workspace than a
 * path needs the next one is taken, AUTODDL_EWORK if none fits.  Tables with K <= 64 (given or built) of at most 64 chains
 * of at least 32 layers take the same layer-parallel scheme on the tiles themselves.
 * Cells must lie in [0, 2^62 / L) so that sums cannot overflow. */
int autoddl_chain_dp(const autoddl_layer* d_layers, int32_t Bp, int32_t L,
                     const autoddl_mesh* mesh, const autoddl_net* net,
                     const int64_t* d_T, void* d_work, size_t work_bytes,
                     int64_t* d_opt_cost, int32_t* d_strategy, void* stream);

/* (a3) Coordinate Descent from S starts per problem.  One sweep visits l = 0..L-1 in order and sets
 * s_l to the smallest-index minimiser of T[l][s_{l-1}][c] + T[l+1][c][s_{l+1}] (s_{-1} = 0, last
 * layer has no second term) using already-updated neighbours; stops after the first sweep that
 * changes nothing or after max_sweeps.  d_sweeps counts sweeps including the final unchanged one.
 * d_init entries must lie in [0, K).  d_T == NULL as in autoddl_chain_dp.  With S >= 32 starts the update of a layer is
 * tabulated once per (left, right) neighbour (from the tiles' factors on 2- / 3-level meshes with d_T == NULL, from the
 * tiles themselves when K <= 64 and d_work holds autoddl_workspace_bytes) and a sweep is one look-up per layer: same
 * trajectory, sweep count and result.  Otherwise, on chains of at least 8 layers and with 1 < max_sweeps < 32768, the
 * sweeps of a start run side by side (sweep k two layers behind sweep k-1: every update reads
 * the operands it reads in the sequential order) -- again the same trajectory, sweep count and result. */
int autoddl_coord_descent(const autoddl_layer* d_layers, int32_t Bp, int32_t L,
                          const autoddl_mesh* mesh, const autoddl_net* net,
                          const int64_t* d_T, void* d_work, size_t work_bytes,
                          const int32_t* d_init, int32_t S, int32_t max_sweeps,
                          int64_t* d_cost, int32_t* d_strategy, int32_t* d_sweeps, void* stream);

/* Metropolis-Hastings sampler on the tables (R19-R22): P(S) ~ exp(-Cost(S) / tau_ps).
 * One chain per (problem, start), nsteps proposals each.  Step t of chain c = p * S + r draws, with rng(n) the
 * n-th output of splitmix64 started at `seed`,
 *   l = rng(4 (c 2^32 + t) + 1) mod L,   s' = rng(.. + 2) mod K,   x = (rng(.. + 3) >> 32) + 1  in [1, 2^32]
 * and accepts s_l <- s' iff dC <= 0 or (dC < 2^45 and tau_ps * neglog_q16(x) >= dC * 2^16), dC = Cost(S_new) -
 * Cost(S_old), neglog_q16(x) = -ln(x / 2^32) in Q16 by 16 shift-and-square steps on a Q62 mantissa, ln 2 =
 * 744261117 / 2^30 (integer only: results are bit-exact).  That is acceptance with probability
 * min(1, P(S_new) / P(S_old)).  Outputs per chain: d_best_cost [Bp][S] the smallest cost seen (start included) and
 * d_best_strategy [Bp][S][L] the first strategy attaining it, d_final_cost / d_final_strategy the last state,
 * d_accepted [Bp][S] the number of accepted proposals.  0 <= tau_ps < 2^40, nsteps >= 0, K <= 256,
 * d_init entries in [0, K). */
int autoddl_metropolis(const int64_t* d_T, int32_t Bp, int32_t L, const autoddl_mesh* mesh,
                       const int32_t* d_init, int32_t S, int32_t nsteps, int64_t tau_ps, uint64_t seed,
                       int64_t* d_best_cost, int32_t* d_best_strategy, int64_t* d_final_cost,
                       int32_t* d_final_strategy, int32_t* d_accepted, void* stream);

/* alpha-beta calibration: least-squares (alpha, beta) of the linear system of Table 2
 *   t_i = A_i alpha + B_i beta  over N timed collectives, d_kind[i] in {0 AllGather, 1 ReduceScatter,
 * 2 AllReduce, 3 AlltoAll}, d_p[i] >= 2 participants, d_bytes[i] message bytes, d_time[i] measured time (any unit):
 * (A, B) = (p-1, (p-1)/p n), (2p-1, 2 (p-1)/p n) for AllReduce, (p-1, n) for AlltoAll.  fp64; d_out[0] = alpha,
 * d_out[1] = beta (time unit per byte).  d_work: >= autoddl_fit_workspace_bytes() bytes, 8-byte aligned.
 * Deterministic (fixed grid and reduction order). */
size_t autoddl_fit_workspace_bytes(void);
int autoddl_fit_alpha_beta(const int32_t* d_kind, const int32_t* d_p, const int64_t* d_bytes, const double* d_time,
                           int64_t N, double* d_out, void* d_work, size_t work_bytes, void* stream);

/* Whole path on DEVICE pointers, one call: (a1) -> (a2) -> (a3).  On a 2-level mesh (K = 36) with at least 296
 * chains (a1), (a2) and the first two sweeps of (a3) for up to 8 starts per chain run as ONE kernel, one warp per chain:
 * every tile is evaluated in factor form in shared memory, written to d_T with coalesced stores and consumed by the
 * chain DP and the CD sweeps from shared memory, so the optimum costs no table read; the CD kernel resumes at sweep 3.
 * Few chains take the kernels of autoddl_chain_dp / autoddl_coord_descent (class-space or layer-parallel DP, look-up CD
 * where they apply); kernels that do not depend on one another then run side by side on two library-owned side
 * streams (created on first use, per host thread and device), ordered by events against `stream`: on return all work
 * is ordered behind `stream` as if it had been launched there.  Results are identical to the three separate calls.
 * The call allocates nothing and synchronises nothing: it can be captured into a CUDA graph and replayed (make one eager
 * call with the same shapes first: it creates the side streams and the device-wide index tables).
 * d_T: [Bp][L][K][K] output, or NULL to keep the tables in d_work (any mesh) -- with d_init == NULL
 * and K = 36 no table is materialised at all.  d_node / d_mask may be NULL.  d_init == NULL skips (a3).
 * d_work: >= autoddl_workspace_bytes(Bp, L, S, mesh). */
int autoddl_search(const autoddl_layer* d_layers, int32_t Bp, int32_t L,
                   const autoddl_mesh* mesh, const autoddl_net* net,
                   int64_t* d_T, int64_t* d_node, uint8_t* d_mask, void* d_work, size_t work_bytes,
                   int64_t* d_opt_cost, int32_t* d_strategy,
                   const int32_t* d_init, int32_t S, int32_t max_sweeps,
                   int64_t* d_cd_cost, int32_t* d_cd_strategy, int32_t* d_cd_sweeps, void* stream);

/* Whole path with HOST inputs and outputs (the end-to-end call): brings h_layers and h_init to the device -- inputs in
 * pinned, device-mapped host memory (cudaHostAlloc / cudaHostRegister) are read by the kernels straight over PCIe, once,
 * overlapped with the table stores; pageable inputs are copied first -- runs (a1) (a2) (a3) in d_work, copies the
 * results back (the optimum and its strategy on an internal side stream while Coordinate Descent still runs),
 * synchronises `stream`: all outputs are complete on return.
 * Any h_* output may be NULL to skip it; h_init NULL skips (a3). */
int autoddl_search_host(const autoddl_layer* h_layers, int32_t Bp, int32_t L,
                        const autoddl_mesh* mesh, const autoddl_net* net,
                        const int32_t* h_init, int32_t S, int32_t max_sweeps,
                        void* d_work, size_t work_bytes,
                        int64_t* h_opt_cost, int32_t* h_strategy,
                        int64_t* h_cd_cost, int32_t* h_cd_strategy, int32_t* h_cd_sweeps, void* stream);

/* (a2) on caller-supplied tables WITHOUT any allocation and without a workspace argument, for callers that cannot call
 * cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it): the layer-parallel chain DP
 * of autoddl_chain_dp for K <= 64 with its scratch -- chunk products, prefix vectors,
 * back-pointers -- in a static device array of AUTODDL_STATIC_SCRATCH_BYTES that every GPU loading the library holds until
 * exit.  Same results as autoddl_chain_dp (same optimum, smallest index on every tie).
 * d_T [Bp][L][K][K] int64 (8-byte aligned), d_opt_cost [Bp] int64, d_strategy [Bp][L] int32: device pointers, owned by
 * the caller.  Accepted: K <= 64, 1 <= Bp <= 64, L >= 32 (AUTODDL_EINVAL otherwise), and
 * autoddl_chain_dp_static_bytes(Bp, L, mesh) <= AUTODDL_STATIC_SCRATCH_BYTES (AUTODDL_EWORK otherwise: use
 * autoddl_chain_dp with a workspace).  Calls no cudaMalloc / cudaFree / allocating routine; asynchronous on `stream`.
 * ALL calls on a device share the one array, which keeps the last call's contents (nothing needs to start at zero):
 * calls that overlap on the GPU -- two streams, two host threads -- race; serialise them. */
#define AUTODDL_STATIC_SCRATCH_BYTES (8u << 20)
int autoddl_chain_dp_static(const int64_t* d_T, int32_t Bp, int32_t L, const autoddl_mesh* mesh,
                            int64_t* d_opt_cost, int32_t* d_strategy, void* stream);
/* Bytes of the static array a call with (Bp, L, mesh) uses; 0 if the arguments are outside the accepted ranges. Host only. */
size_t autoddl_chain_dp_static_bytes(int32_t Bp, int32_t L, const autoddl_mesh* mesh);

/* Best of the Coordinate Descent starts ("records the best strategy"): for every problem p the smallest
 * d_cost[p][s] over s = 0..S-1 and the smallest s attaining it.  d_cost [Bp][S] int64, d_best_cost [Bp] int64,
 * d_best_start [Bp] int32: device pointers, 8 / 4-byte aligned; Bp, S >= 1.  Asynchronous on `stream`. */
int autoddl_best_of_starts(const int64_t* d_cost, int32_t Bp, int32_t S, int64_t* d_best_cost, int32_t* d_best_start,
                           void* stream);

/* ---- Pipeline stages ("consecutive layers form a pipeline stage", 1F1B, Table 3 "Opt.
 * Stages"; R27).  ONE chain of L layers.  A stage is a contiguous segment [a, b) of the chain on its own
 * sub-mesh (the mesh with 1 / stages of the nodes); d_T / d_node / d_mask are the outputs of autoddl_build_tables for the
 * chain ON THAT SUB-MESH.  The stage COST MODEL below is this library's reading: the paper prints none.
 *
 * autoddl_segment_optima: d_tri [L][L + 1] int64, d_tri[a][b] = C(a, b) = the optimum over all K^(b-a) strategies of the
 *   segment [a, b) as a chain of its own whose first layer has no producer (f_a[j] = node[a][j] + 2^50 [mask[a][j] == 0]);
 *   -1 for a >= b.  One pass over the tables for all L (L + 1) / 2 segments (min-plus products of 16 starts at a time).
 * autoddl_stage_transfer: d_xfer [L] int64, d_xfer[b] = 2 m (alpha_inter + ceil(in_rows_b in_cols_b act_bytes_b / q)
 *   beta_inter): the input of layer b, split over the q devices of the sub-mesh, crosses the network point to point
 *    forward and backward once per micro-batch (m = net.micro_batches); d_xfer[0] = 0.
 * autoddl_pipeline_partition: the best `stages` contiguous non-empty segments; stage cost c(a, b) = C(a, b) + xfer[a] +
 *   [b < L] xfer[b]; objective 0 = sum of the stage costs, 1 = max (the slowest stage paces a 1F1B pipeline).
 *   g_1[b] = c(0, b); g_k[b] = min_a comb(g_{k-1}[a], c(a, b)), smallest a on ties; d_value [1] = g_stages[L];
 *   d_cuts [stages + 1] by back-tracking (d_cuts[0] = 0, d_cuts[stages] = L).  d_work >= autoddl_pipeline_workspace_bytes.
 * autoddl_segment_strategies: per stage k the optimum strategy of [d_cuts[k], d_cuts[k + 1]) (smallest index on every
 *   tie, as autoddl_chain_dp): d_seg_cost [stages] = C(.,.), d_strategy [L].  d_cuts is read on the device: no host
 *   synchronisation between the partition and the strategies.  d_work >= autoddl_pipeline_workspace_bytes.
 * All pointers are device pointers (8-byte aligned for int64, 4 for int32, d_work 256); asynchronous on `stream`.
 * The outer enumeration over stage counts (build the tables on every candidate sub-mesh, partition, compare) is the
 * caller's loop. */
size_t autoddl_pipeline_workspace_bytes(int32_t L, int32_t K, int32_t stages);
int autoddl_segment_optima(const int64_t* d_T, const int64_t* d_node, const uint8_t* d_mask, int32_t L,
                           const autoddl_mesh* mesh, int64_t* d_tri, void* stream);
int autoddl_stage_transfer(const autoddl_layer* d_layers, int32_t L, const autoddl_mesh* mesh, const autoddl_net* net,
                           int64_t* d_xfer, void* stream);
int autoddl_pipeline_partition(const int64_t* d_tri, const int64_t* d_xfer, int32_t L, int32_t stages, int32_t objective,
                               void* d_work, size_t work_bytes, int64_t* d_value, int32_t* d_cuts, void* stream);
int autoddl_segment_strategies(const int64_t* d_T, const int64_t* d_node, const uint8_t* d_mask, int32_t L,
                               const autoddl_mesh* mesh, const int32_t* d_cuts, int32_t stages, void* d_work, size_t work_bytes,
                               int64_t* d_seg_cost, int32_t* d_strategy, void* stream);

/* Plain device-to-device copy kernel (int4 grid-stride), used by bench.py to measure the HBM
 * copy bandwidth in the same run as the kernels above.  bytes must be a multiple of 16. */
int autoddl_copy_probe(const void* d_src, void* d_dst, size_t bytes, void* stream);

/* Store-only probe with the address pattern of the fused table writer of autoddl_search: one warp per chain writes the
 * chain's L tiles of K x K int64 cells in order with 16-byte streaming stores (no arithmetic; the cells are overwritten
 * with filler).  bench.py times it in the same run: the ceiling of that write pattern, next to the copy bandwidth.
 * d_T: [Bp][L][K][K] int64 device buffer, 16-byte aligned; K * K even. */
int autoddl_store_probe(int64_t* d_T, int32_t Bp, int32_t L, int32_t K, void* stream);

/* Profiling hook (used by bench.py for the per-kernel split of the one-call path): the next autoddl_search /
 * autoddl_search_host call of this thread records `cuda_event` (a cudaEvent_t, NULL to cancel) on its stream after
 * the tables + chain DP and before Coordinate Descent.  One shot. */
int autoddl_profile_mark(void* cuda_event);

/* Number of kernel launches issued by this library in the calling thread since load (for bench.py's
 * gpu_launches). */
int64_t autoddl_launch_count(void);

/* Text of the last error in the calling thread ("" if none). */
const char* autoddl_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
