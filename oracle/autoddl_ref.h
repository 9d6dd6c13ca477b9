/*
 * oracle/autoddl_ref.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU restatement of the AutoDDL strategy-search
 * hot path (arxiv 2301.06813), written from PAPER.md and the readings listed
 * in DESIGN.md section 3 ("Readings").  It shares no code, header, table or
 * helper with the CUDA path under paper_2301_06813_b200/csrc; the struct
 * layouts below are restated here on purpose.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may load it.
 *
 * All costs are int64 picoseconds.  All pointers are HOST pointers.
 *
 * Parity status (see DESIGN.md section 4 "Pins"):
 *   collectives (Table 2)        pinned  (hand values, identities)
 *   reshard path                pinned  (paper's 15 GB example, hand cells on divisible AND ragged dims:
 *                                                  level order, message size before / after, scatter axis, fwd != bwd)
 *   weight-gradient sync        pinned  (data-parallel closed form, ragged local weight by hand)
 *   memory feasibility          PARITY UNPINNED (paper gives no formula; ours: hand value + boundaries)
 *   chain DP optimum (PAPER.md:225 exhaustive)     pinned  (brute force over K^L)
 *   coordinate descent          pinned by properties (1-opt, monotone, DP <= CD)
 *   folded factorisation space pinned  (equal, cell by cell, to the canonical signatures of the prime-
 *                                                  sub-level encoding on every machine both express; decode order by
 *                                                  enumeration; data-parallel closed form on 2^6 .. 2^8 nodes)
 *   four / five mesh levels    pinned  (size-1 levels reproduce the three-level tables, decode order,
 *                                                  data-parallel closed form, intra-node gather, brute force at K = 81)
 *   pipeline stages         segment optima and the partition pinned (one stage = the chain DP,
 *                                                  brute force over strategies and over cut sets); the stage COST MODEL
 *                                                  (transfer term, sum / max objective) is PARITY UNPINNED: the paper prints none
 *   Metropolis-Hastings         pinned  (Boltzmann stationary law on enumerable chains, greedy and
 *                                                  hot limits, integer -ln against libm, replay of a hand-checked chain)
 */
#ifndef AUTODDL_REF_H
#define AUTODDL_REF_H

#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* tensor states per mesh level, PAPER.md:140,160 (Split axis 0 / axis 1, Broadcast, Partial-sum) */
enum { REF_S0 = 0, REF_S1 = 1, REF_B = 2, REF_P = 3 };
/* layer kinds */
enum { REF_GEMM = 0, REF_ATTN = 1 };

typedef struct {
  int64_t M, Kd, N;          /* O[M,N] = I[M,Kd] * W[Kd,N] */
  int64_t in_rows, in_cols;  /* activation resharded into this layer */
  int32_t kind;
  int32_t act_bytes;
  int32_t wgrad_bytes;
  int32_t wstate_bytes;
  int32_t max_split_rows;
  int32_t max_split_cols;
} ref_layer;                 /* 64 bytes */

/* link[d]: bit 0 = 0 intra / 1 inter; bits 8..13 = allowed signature rows of the level (bit g = row g; 0 = all six);
 * bit 14 of link[0] = FOLDED factorisation space (R28): rows {0,1,2} on every level, and inside every group of
 * consecutive levels with equal size and link class only the sorted digit strings 0..0 1..1 2..2 are signatures -- the
 * paper's ordered factorisations p = p0 p1 p2 with (nodes, GPUs) tuples.  ndim up to 8 when folded. */
#define REF_MAX_LEVELS 8
#define REF_FOLD 0x4000
typedef struct { int32_t ndim; int32_t size[REF_MAX_LEVELS]; int32_t link[REF_MAX_LEVELS]; } ref_mesh;
/* micro_batches: gradient accumulation: the activation redistributions run once per micro-batch,
 * the weight-gradient synchronisation once per mini-batch; 0 or 1 = no accumulation (R25) */
typedef struct { int64_t alpha_ps[2]; int64_t beta_ps_per_byte[2]; int64_t mem_cap_bytes; int64_t micro_batches; } ref_net;

#define REF_PEN ((int64_t)1 << 50)

/* signatures per layer: 6^ndim for ndim <= 3; for ndim = 4, 5 the product of the levels' allowed-row counts
 * (<= 256, else -1): there the signature index is a mixed-radix number over the allowed rows only (R26);
 * folded (R28): the product over the groups of equal levels of C(n_g + 2, 2) (<= 256), group 0 most significant, inside
 * a group the sorted strings in increasing lexicographic order */
int autoddl_ref_num_signatures(const ref_mesh* mesh);

/* Table 2. which: 0 AllGather, 1 ReduceScatter, 2 AllReduce, 3 AlltoAll */
int64_t autoddl_ref_collective(int which, int64_t n_bytes, int64_t p, int64_t alpha, int64_t beta);

/* local element count of an R x C tensor in state vector st[ndim] (Fig. 5) */
int64_t autoddl_ref_local_size(int64_t R, int64_t C, const int32_t* st, const ref_mesh* mesh);

/* (I, W, O) state vectors of signature sig for a layer kind; returns 1 if valid, 0 if not */
int autoddl_ref_sig_states(int kind, int sig, const ref_mesh* mesh, int32_t* I, int32_t* W, int32_t* O);

/* forward redistribution cost a -> b of a rows x cols tensor with eb bytes/element */
int64_t autoddl_ref_reshard(int64_t rows, int64_t cols, int64_t eb, const int32_t* a, const int32_t* b,
                            const ref_mesh* mesh, const ref_net* net);

/* edge / node / feasibility of one cell, straight from the definitions */
int64_t autoddl_ref_edge_cost(const ref_layer* prev, const ref_layer* cur, int i, int j,
                              const ref_mesh* mesh, const ref_net* net);
int64_t autoddl_ref_node_cost(const ref_layer* cur, int j, const ref_mesh* mesh, const ref_net* net);
int     autoddl_ref_feasible(const ref_layer* cur, int j, int32_t L, const ref_mesh* mesh, const ref_net* net);
int64_t autoddl_ref_layer_mem(const ref_layer* cur, int j, const ref_mesh* mesh);

/* (a1) T[Bp][L][K][K], node[Bp][L][K], mask[Bp][L][K]; node/mask may be NULL */
int autoddl_ref_build_tables(const ref_layer* layers, int32_t Bp, int32_t L, const ref_mesh* mesh,
                             const ref_net* net, int64_t* T, int64_t* node, uint8_t* mask);

/* Cost(S) = sum_l T[l][s_{l-1}][s_l], s_{-1} = 0 (one problem) */
int64_t autoddl_ref_chain_cost(const int64_t* T, int32_t L, int32_t K, const int32_t* s);

/* (a2) exact min-plus chain DP, lowest-index tie-breaks */
int autoddl_ref_chain_dp(const int64_t* T, int32_t Bp, int32_t L, int32_t K,
                         int64_t* opt_cost, int32_t* strategy);

/* exhaustive enumeration of all K^L strategies of one problem (the paper's "exhaustive search") */
int autoddl_ref_brute_force(const int64_t* T, int32_t L, int32_t K, int64_t* opt_cost, int32_t* strategy);

/* (a3) coordinate descent; trace (optional) receives Cost(s) after every layer update:
 * trace[Bp][S][max_sweeps][L], unused tail untouched */
int autoddl_ref_coord_descent(const int64_t* T, int32_t Bp, int32_t L, int32_t K,
                              const int32_t* init, int32_t S, int32_t max_sweeps,
                              int64_t* cost, int32_t* strategy, int32_t* sweeps, int64_t* trace);

/* best of the starts of every problem: smallest cost, then smallest start index */
int autoddl_ref_best_of_starts(const int64_t* cost, int32_t Bp, int32_t S, int64_t* best_cost, int32_t* best_start);

/* ---- pipeline stages (R27) ------------------------------------------------------------
 * tri[a * (L + 1) + b] = optimum of the segment [a, b) as its own chain whose first layer has no producer (-1 elsewhere) */
int autoddl_ref_segment_optima(const int64_t* T, const int64_t* node, const uint8_t* mask, int32_t L, int32_t K, int64_t* tri);
/* xfer[b] = 2 m (alpha_inter + ceil(bytes of layer b's input / devices of the mesh) beta_inter), xfer[0] = 0 */
int autoddl_ref_stage_transfer(const ref_layer* layers, int32_t L, const ref_mesh* mesh, const ref_net* net, int64_t* xfer);
/* best `stages` contiguous segments; objective 0 = sum of the stage costs, 1 = max; cuts[stages + 1] */
int autoddl_ref_pipeline_partition(const int64_t* tri, const int64_t* xfer, int32_t L, int32_t stages, int32_t objective,
                                   int64_t* value, int32_t* cuts);
/* per-segment optimum strategies under given cuts: seg_cost[stages], strategy[L] */
int autoddl_ref_segment_strategies(const int64_t* T, const int64_t* node, const uint8_t* mask, int32_t L, int32_t K,
                                   const int32_t* cuts, int32_t stages, int64_t* seg_cost, int32_t* strategy);

/* ---- Metropolis-Hastings sampler (R19-R22) --------------------------------
 * n-th output (n >= 1) of splitmix64 started at `seed`: the counter-based generator both sides implement. */
uint64_t autoddl_ref_rng(uint64_t seed, uint64_t n);
/* floor-style fixed point -ln(x / 2^32) * 2^16 for x in [1, 2^32], by integer shift-and-square (R21) */
int64_t autoddl_ref_neglog_q16(uint64_t x);
/* One chain per (problem, start), nsteps proposals each.  Step t of chain c = p * S + r draws
 *   l = rng(4 (c 2^32 + t) + 1) mod L,  s' = rng(.. + 2) mod K,  x = (rng(.. + 3) >> 32) + 1
 * and accepts the move s_l <- s' iff dC <= 0 or (dC < 2^45 and tau * neglog_q16(x) >= dC * 2^16), i.e. with
 * probability min(1, exp(-dC / tau)) = min(1, P(S_new) / P(S_old)) for P(S) ~ exp(-Cost(S) / tau).
 * Outputs per chain: smallest cost seen (first time attained) and its strategy, the final strategy and cost,
 * the number of accepted proposals.  trace (optional) [Bp][S][nsteps] = cost after every step. */
int autoddl_ref_metropolis(const int64_t* T, int32_t Bp, int32_t L, int32_t K,
                           const int32_t* init, int32_t S, int32_t nsteps, int64_t tau_ps, uint64_t seed,
                           int64_t* best_cost, int32_t* best_strategy, int64_t* final_cost, int32_t* final_strategy,
                           int32_t* accepted, int64_t* trace);

#ifdef __cplusplus
}
#endif
#endif
