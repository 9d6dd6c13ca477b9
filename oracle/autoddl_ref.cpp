// oracle/autoddl_ref.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see autoddl_ref.h).
//
// Plain single-threaded C++.  Every function follows one passage of PAPER.md
// (cited) in the reading DESIGN.md section 3 fixes (R1..R18).  No blocking, no
// factorisation of the K x K table into state tables, no caching: each cell of
// T is evaluated from scratch from its definition.
//
// Build: g++ -O2 -std=c++17 -shared -fPIC oracle/autoddl_ref.cpp -o oracle/libautoddl_ref.so
#include "autoddl_ref.h"

#include <cstdint>
#include <climits>
#include <vector>

namespace {

inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ---- R1: signature table --------------------------------------------------
// Rows 0..2 are the three factors of the paper's SBP matmul (PAPER.md:193:
// I=(S0,B,S1), W=(B,S1,S0), O=(S0,S1,P)); row 3 replicates everything; rows 4
// and 5 let a partial-sum operand pass through the (linear) matmul.
const int32_t GEMM_I[6] = {REF_S0, REF_B,  REF_S1, REF_B, REF_P, REF_B};
const int32_t GEMM_W[6] = {REF_B,  REF_S1, REF_S0, REF_B, REF_B, REF_P};
const int32_t GEMM_O[6] = {REF_S0, REF_S1, REF_P,  REF_B, REF_P, REF_P};
// Attention has no weight and is not linear in a partial-sum input: it may be
// split over rows (batch), over columns (heads) or replicated.
const int32_t ATTN_IO[6]    = {REF_S0, REF_S1, -1, REF_B, -1, -1};

inline int ipow6(int d) { int k = 1; for (int t = 0; t < d; ++t) k *= 6; return k; }

// rows a level admits: bits 8..13 of link[d], bit g = row g; 0 = all six (R24)
inline int level_allow(const ref_mesh* mesh, int d) {
  const int a = (mesh->link[d] >> 8) & 0x3f;
  return a ? a : 0x3f;
}
inline int level_nrows(const ref_mesh* mesh, int d) {
  int n = 0;
  for (int g = 0; g < 6; ++g) n += (level_allow(mesh, d) >> g) & 1;
  return n;
}

inline bool folded(const ref_mesh* mesh) { return (mesh->link[0] & REF_FOLD) != 0; }

// R28: groups of the folded space = maximal runs of consecutive levels with equal size and link class.  Returns the
// number of groups; first[g] = first level of group g, len[g] = its number of levels.
inline int fold_groups(const ref_mesh* mesh, int* first, int* len) {
  int ng = 0;
  for (int d = 0; d < mesh->ndim; ++d) {
    if (d > 0 && mesh->size[d] == mesh->size[d - 1] && (mesh->link[d] & 1) == (mesh->link[d - 1] & 1)) {
      ++len[ng - 1];
    } else {
      first[ng] = d;
      len[ng] = 1;
      ++ng;
    }
  }
  return ng;
}
inline int fold_radix(int n) { return (n + 2) * (n + 1) / 2; }       // sorted strings of length n over {0,1,2}

// per-level row of level d in signature index j, level 0 most significant.
// ndim <= 3: j is a base-6 number over all six rows (a disallowed row makes the signature infeasible, R24).
// ndim  > 3: j is a mixed-radix number over the ALLOWED rows only (R26): the digit x of level d is the x-th allowed
//            row of that level in increasing order; the radix of level d is its number of allowed rows.
// folded (R28): j is a mixed-radix number over the groups (group 0 most significant); the digit x of a group of n levels
//            names the x-th sorted string 0^n0 1^n1 2^n2 (n0 + n1 + n2 = n) in increasing lexicographic order, i.e.
//            n0 = n, n-1, .. and, for equal n0, n1 descending; level t of the group has row 0 / 1 / 2 accordingly.
inline int sig_digit(int j, int d, const ref_mesh* mesh) {
  const int D = mesh->ndim;
  if (folded(mesh)) {
    int first[REF_MAX_LEVELS], len[REF_MAX_LEVELS];
    const int ng = fold_groups(mesh, first, len);
    int g = 0;
    while (g + 1 < ng && first[g + 1] <= d) ++g;                     // the group of level d
    int div = 1;
    for (int t = g + 1; t < ng; ++t) div *= fold_radix(len[t]);
    int x = (j / div) % fold_radix(len[g]);
    const int n = len[g], t = d - first[g];
    for (int n0 = n; n0 >= 0; --n0)
      for (int n1 = n - n0; n1 >= 0; --n1) {
        if (x == 0) return t < n0 ? 0 : (t < n0 + n1 ? 1 : 2);
        --x;
      }
    return -1;                                // not reached
  }
  if (D <= 3) {
    int div = 1;
    for (int t = 0; t < D - 1 - d; ++t) div *= 6;
    return (j / div) % 6;
  }
  int div = 1;
  for (int t = d + 1; t < D; ++t) div *= level_nrows(mesh, t);
  int x = (j / div) % level_nrows(mesh, d);
  for (int g = 0; g < 6; ++g)
    if ((level_allow(mesh, d) >> g) & 1) {
      if (x == 0) return g;
      --x;
    }
  return -1;                                  // not reached
}

inline int32_t dual_state(int32_t s) {   // R9: S0->S0, S1->S1, B->P, P->B
  if (s == REF_B) return REF_P;
  if (s == REF_P) return REF_B;
  return s;
}

}  // namespace

extern "C" int autoddl_ref_num_signatures(const ref_mesh* mesh) {
  if (!mesh || mesh->ndim < 1 || mesh->ndim > REF_MAX_LEVELS) return -1;
  if (folded(mesh)) {                           // R28: product over the groups of the number of ordered factorisations
    int first[REF_MAX_LEVELS], len[REF_MAX_LEVELS];
    const int ng = fold_groups(mesh, first, len);
    int64_t k = 1;
    for (int g = 0; g < ng; ++g) k *= fold_radix(len[g]);
    return k <= 256 ? (int)k : -1;
  }
  if (mesh->ndim > 5) return -1;                // more than five levels only in the folded space
  if (mesh->ndim <= 3) return ipow6(mesh->ndim);
  int64_t k = 1;                              // R26: product of the levels' allowed-row counts, at most 256
  for (int d = 0; d < mesh->ndim; ++d) k *= level_nrows(mesh, d);
  return k <= 256 ? (int)k : -1;
}

extern "C" int autoddl_ref_sig_states(int kind, int sig, const ref_mesh* mesh,
                                      int32_t* I, int32_t* W, int32_t* O) {
  const int D = mesh->ndim;
  int valid = 1;
  for (int d = 0; d < D; ++d) {
    const int g = sig_digit(sig, d, mesh);
    if (kind == REF_GEMM) {
      I[d] = GEMM_I[g]; W[d] = GEMM_W[g]; O[d] = GEMM_O[g];
    } else {
      if (ATTN_IO[g] < 0) { valid = 0; I[d] = W[d] = O[d] = REF_B; }
      else { I[d] = ATTN_IO[g]; O[d] = ATTN_IO[g]; W[d] = REF_B; }
    }
  }
  return valid;
}

// ---- R2: local size (Fig. 5: S splits an axis, B and P keep the full extent)
extern "C" int64_t autoddl_ref_local_size(int64_t R, int64_t C, const int32_t* st, const ref_mesh* mesh) {
  int64_t f0 = 1, f1 = 1;
  for (int d = 0; d < mesh->ndim; ++d) {
    if (st[d] == REF_S0) f0 *= mesh->size[d];
    if (st[d] == REF_S1) f1 *= mesh->size[d];
  }
  return ceil_div(R, f0) * ceil_div(C, f1);
}

// ---- R3: Table 2, n in bytes, (p-1)/p*n evaluated as (p-1)*ceil(n/p)
extern "C" int64_t autoddl_ref_collective(int which, int64_t n, int64_t p, int64_t alpha, int64_t beta) {
  if (p <= 1) return 0;                       // R3/A3: a group of one does not communicate
  const int64_t sh = ceil_div(n, p);
  switch (which) {
    case 0:                                   // AllGather      (p-1)a + (p-1)/p n b
    case 1:                                   // ReduceScatter  same row of Table 2
      return (p - 1) * alpha + (p - 1) * sh * beta;
    case 2:                                   // AllReduce      (2p-1)a + 2 (p-1)/p n b
      return (2 * p - 1) * alpha + 2 * (p - 1) * sh * beta;
    case 3:                                   // AlltoAll       (p-1)a + n b
      return (p - 1) * alpha + n * beta;
  }
  return -1;
}

// ---- R4: forward redistribution a -> b (reduce-scatter, all-to-all, all-gather)
extern "C" int64_t autoddl_ref_reshard(int64_t rows, int64_t cols, int64_t eb,
                                       const int32_t* a, const int32_t* b,
                                       const ref_mesh* mesh, const ref_net* net) {
  const int D = mesh->ndim;
  int32_t cur[REF_MAX_LEVELS];
  for (int d = 0; d < D; ++d) cur[d] = a[d];
  int64_t cost = 0;

  // Ph0 slice (free): a replicated level that must become split just keeps its slice
  for (int d = 0; d < D; ++d)
    if (cur[d] == REF_B && (b[d] == REF_S0 || b[d] == REF_S1)) cur[d] = b[d];

  // Ph1 reduce, innermost level first: P -> S by reduce-scatter ("(S0,S1,P) -> (S0,S1*p2)")
  for (int d = D - 1; d >= 0; --d)
    if (cur[d] == REF_P && b[d] != REF_P) {
      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // RS input size (Table 2 caption)
      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)
      cost += autoddl_ref_collective(1, n, mesh->size[d], net->alpha_ps[c], net->beta_ps_per_byte[c]);
      cur[d] = (b[d] == REF_B) ? REF_S1 : b[d];
    }

  // Ph2 all-to-all, innermost first: change of split axis
  for (int d = D - 1; d >= 0; --d) {
    const bool cs = (cur[d] == REF_S0 || cur[d] == REF_S1);
    const bool bs = (b[d] == REF_S0 || b[d] == REF_S1);
    if (cs && bs && cur[d] != b[d]) {
      cur[d] = b[d];
      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // output size
      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)
      cost += autoddl_ref_collective(3, n, mesh->size[d], net->alpha_ps[c], net->beta_ps_per_byte[c]);
    }
  }

  // Ph3 gather, outermost level first: S -> B by all-gather
  for (int d = 0; d < D; ++d)
    if ((cur[d] == REF_S0 || cur[d] == REF_S1) && b[d] == REF_B) {
      cur[d] = REF_B;
      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // output size
      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)
      cost += autoddl_ref_collective(0, n, mesh->size[d], net->alpha_ps[c], net->beta_ps_per_byte[c]);
    }

  // Ph4 fill (free): a value becomes a partial sum by zero-padding
  for (int d = 0; d < D; ++d)
    if (b[d] == REF_P) cur[d] = REF_P;

  for (int d = 0; d < D; ++d)
    if (cur[d] != b[d]) return -1;            // cannot happen; caught by tests
  return cost;
}

// ---- R5: edge cost = forward redistribution + backward redistribution (PAPER.md:197
// "in both the forward path and the backward path").  The tensor is the consumer's input.
extern "C" int64_t autoddl_ref_edge_cost(const ref_layer* prev, const ref_layer* cur, int i, int j,
                                         const ref_mesh* mesh, const ref_net* net) {
  int32_t Ii[REF_MAX_LEVELS], Wi[REF_MAX_LEVELS], Oi[REF_MAX_LEVELS], Ij[REF_MAX_LEVELS], Wj[REF_MAX_LEVELS], Oj[REF_MAX_LEVELS];
  const int vi = autoddl_ref_sig_states(prev->kind, i, mesh, Ii, Wi, Oi);
  const int vj = autoddl_ref_sig_states(cur->kind, j, mesh, Ij, Wj, Oj);
  if (!vi || !vj) return 0;
  int32_t da[REF_MAX_LEVELS], db[REF_MAX_LEVELS];
  for (int d = 0; d < mesh->ndim; ++d) { da[d] = dual_state(Oi[d]); db[d] = dual_state(Ij[d]); }
  const int64_t fwd = autoddl_ref_reshard(cur->in_rows, cur->in_cols, cur->act_bytes, Oi, Ij, mesh, net);
  const int64_t bwd = autoddl_ref_reshard(cur->in_rows, cur->in_cols, cur->act_bytes, db, da, mesh, net);
  return fwd + bwd;
}

// ---- R6: weight-gradient synchronisation: every level on which W is
// replicated (B) all-reduces the local weight gradient.
extern "C" int64_t autoddl_ref_node_cost(const ref_layer* cur, int j, const ref_mesh* mesh, const ref_net* net) {
  if (cur->kind != REF_GEMM) return 0;
  int32_t I[REF_MAX_LEVELS], W[REF_MAX_LEVELS], O[REF_MAX_LEVELS];
  if (!autoddl_ref_sig_states(cur->kind, j, mesh, I, W, O)) return 0;
  const int64_t nw = autoddl_ref_local_size(cur->Kd, cur->N, W, mesh);
  int64_t v = 0;
  for (int d = 0; d < mesh->ndim; ++d)
    if (W[d] == REF_B) {
      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)
      v += autoddl_ref_collective(2, nw * cur->wgrad_bytes, mesh->size[d], net->alpha_ps[c], net->beta_ps_per_byte[c]);
    }
  return v;
}

// ---- R7: per-device memory of one layer under signature j (PARITY UNPINNED: PAPER.md:221-223
// uses a OneFlow CPU dry run and prints no formula; this one is ours).
extern "C" int64_t autoddl_ref_layer_mem(const ref_layer* cur, int j, const ref_mesh* mesh) {
  int32_t I[REF_MAX_LEVELS], W[REF_MAX_LEVELS], O[REF_MAX_LEVELS];
  if (!autoddl_ref_sig_states(cur->kind, j, mesh, I, W, O)) return 0;
  int64_t mem = 0;
  if (cur->kind == REF_GEMM) mem += autoddl_ref_local_size(cur->Kd, cur->N, W, mesh) * cur->wstate_bytes;
  mem += (autoddl_ref_local_size(cur->in_rows, cur->in_cols, I, mesh) +
          autoddl_ref_local_size(cur->M, cur->N, O, mesh)) * cur->act_bytes;
  return mem;
}

extern "C" int autoddl_ref_feasible(const ref_layer* cur, int j, int32_t L, const ref_mesh* mesh, const ref_net* net) {
  int32_t I[REF_MAX_LEVELS], W[REF_MAX_LEVELS], O[REF_MAX_LEVELS];
  if (!autoddl_ref_sig_states(cur->kind, j, mesh, I, W, O)) return 0;
  // R24: a level may restrict its signature rows (bits 8..13 of link[d], 0 = all six).  Rows {0,1,2} on every level
  // of a mesh refined into prime sub-levels is the paper's own factorisation space.
  // (with more than three levels the signature index runs over allowed rows only, R26: nothing to exclude)
  for (int d = 0; d < mesh->ndim; ++d)
    if (!folded(mesh) && !((level_allow(mesh, d) >> sig_digit(j, d, mesh)) & 1)) return 0;   // (folded: rows 0..2 by construction)
  int64_t rowsplit = 1, colsplit = 1;
  for (int d = 0; d < mesh->ndim; ++d) {
    if (I[d] == REF_S0 || O[d] == REF_S0) rowsplit *= mesh->size[d];
    if (O[d] == REF_S1) colsplit *= mesh->size[d];
  }
  if (rowsplit > cur->max_split_rows) return 0;      // PAPER.md:189 "constraints on input split dimensions"
  if (colsplit > cur->max_split_cols) return 0;
  if (net->mem_cap_bytes != 0 && autoddl_ref_layer_mem(cur, j, mesh) > net->mem_cap_bytes / L) return 0;
  return 1;
}

// ---- R8: the table.  T[l][i][j] = E(l,i,j) + V(l,j) + PEN*[not feasible(l,j)], E(0,.,.) = 0.
extern "C" int autoddl_ref_build_tables(const ref_layer* layers, int32_t Bp, int32_t L, const ref_mesh* mesh,
                                        const ref_net* net, int64_t* T, int64_t* node, uint8_t* mask) {
  if (!layers || !mesh || !net || !T || Bp < 1 || L < 1) return -1;
  const int K = autoddl_ref_num_signatures(mesh);
  if (K < 0) return -1;
  for (int64_t p = 0; p < Bp; ++p)
    for (int64_t l = 0; l < L; ++l) {
      const ref_layer* cur = &layers[p * L + l];
      const ref_layer* prev = (l > 0) ? &layers[p * L + l - 1] : nullptr;
      int64_t* tile = T + ((p * L + l) * K) * K;
      for (int j = 0; j < K; ++j) {
        const int64_t v = autoddl_ref_node_cost(cur, j, mesh, net);
        const int ok = autoddl_ref_feasible(cur, j, L, mesh, net);
        if (node) node[(p * L + l) * K + j] = v;
        if (mask) mask[(p * L + l) * K + j] = (uint8_t)ok;
        for (int i = 0; i < K; ++i) {
          const int64_t e = prev ? autoddl_ref_edge_cost(prev, cur, i, j, mesh, net) : 0;
          // R25: redistributions once per micro-batch, weight-gradient synchronisation once per mini-batch
          const int64_t m = net->micro_batches > 1 ? net->micro_batches : 1;
          tile[(int64_t)i * K + j] = m * e + v + (ok ? 0 : REF_PEN);
        }
      }
    }
  return 0;
}

// ---- R8: Cost(S) = sum_l T[l][s_{l-1}][s_l], s_{-1} := 0  ("a sequence of collectives")
extern "C" int64_t autoddl_ref_chain_cost(const int64_t* T, int32_t L, int32_t K, const int32_t* s) {
  int64_t c = 0;
  int32_t prev = 0;
  for (int32_t l = 0; l < L; ++l) {
    c += T[((int64_t)l * K + prev) * K + s[l]];
    prev = s[l];
  }
  return c;
}

// ---- R9: exact optimum by min-plus DP over the layered graph; smallest index wins every tie.
extern "C" int autoddl_ref_chain_dp(const int64_t* T, int32_t Bp, int32_t L, int32_t K,
                                    int64_t* opt_cost, int32_t* strategy) {
  if (!T || !opt_cost || !strategy || Bp < 1 || L < 1 || K < 1) return -1;
  std::vector<int64_t> f(K), g(K);
  std::vector<int32_t> bp((size_t)L * K);
  for (int64_t p = 0; p < Bp; ++p) {
    const int64_t* Tp = T + p * L * K * K;
    for (int j = 0; j < K; ++j) f[j] = Tp[j];                       // f_0[j] = T[0][0][j]
    for (int32_t l = 1; l < L; ++l) {
      const int64_t* tile = Tp + (int64_t)l * K * K;
      for (int j = 0; j < K; ++j) {
        int64_t best = f[0] + tile[j];
        int32_t arg = 0;
        for (int i = 1; i < K; ++i) {
          const int64_t v = f[i] + tile[(int64_t)i * K + j];
          if (v < best) { best = v; arg = i; }                      // strict: smallest i kept
        }
        g[j] = best;
        bp[(size_t)l * K + j] = arg;
      }
      f.swap(g);
    }
    int32_t js = 0;
    for (int j = 1; j < K; ++j) if (f[j] < f[js]) js = j;
    opt_cost[p] = f[js];
    int32_t* s = strategy + p * L;
    s[L - 1] = js;
    for (int32_t l = L - 1; l >= 1; --l) s[l - 1] = bp[(size_t)l * K + s[l]];
  }
  return 0;
}

// ---- exhaustive search: odometer over all K^L strategies of one problem;
// the first strategy in lexicographic order attaining the minimum is returned.
extern "C" int autoddl_ref_brute_force(const int64_t* T, int32_t L, int32_t K,
                                       int64_t* opt_cost, int32_t* strategy) {
  if (!T || !opt_cost || !strategy || L < 1 || K < 1) return -1;
  std::vector<int32_t> s(L, 0);
  int64_t best = -1;
  for (;;) {
    const int64_t c = autoddl_ref_chain_cost(T, L, K, s.data());
    if (best < 0 || c < best) { best = c; for (int l = 0; l < L; ++l) strategy[l] = s[l]; }
    int l = L - 1;
    while (l >= 0 && ++s[l] == K) { s[l] = 0; --l; }
    if (l < 0) break;
  }
  *opt_cost = best;
  return 0;
}

// ---- R10: coordinate descent.  One update: S[l] = argmin over s_l of Cost(S)
// with all other layers fixed.  Only the two table entries touching s_l depend on it.
extern "C" int autoddl_ref_coord_descent(const int64_t* T, int32_t Bp, int32_t L, int32_t K,
                                         const int32_t* init, int32_t S, int32_t max_sweeps,
                                         int64_t* cost, int32_t* strategy, int32_t* sweeps, int64_t* trace) {
  if (!T || !init || !cost || !strategy || !sweeps || Bp < 1 || L < 1 || K < 1 || S < 1 || max_sweeps < 1) return -1;
  std::vector<int32_t> s(L);
  for (int64_t p = 0; p < Bp; ++p) {
    const int64_t* Tp = T + p * L * K * K;
    for (int64_t r = 0; r < S; ++r) {
      for (int l = 0; l < L; ++l) s[l] = init[(p * S + r) * L + l];
      int32_t nsweeps = 0;
      for (;;) {
        bool changed = false;
        for (int32_t l = 0; l < L; ++l) {
          const int32_t left = (l > 0) ? s[l - 1] : 0;
          int64_t best = 0;
          int32_t arg = -1;
          for (int c = 0; c < K; ++c) {
            int64_t g = Tp[((int64_t)l * K + left) * K + c];
            if (l < L - 1) g += Tp[((int64_t)(l + 1) * K + c) * K + s[l + 1]];
            if (arg < 0 || g < best) { best = g; arg = c; }
          }
          if (arg != s[l]) { s[l] = arg; changed = true; }
          if (trace) trace[(((p * S + r) * max_sweeps) + nsweeps) * L + l] = autoddl_ref_chain_cost(Tp, L, K, s.data());
        }
        ++nsweeps;
        if (!changed || nsweeps >= max_sweeps) break;
      }
      cost[p * S + r] = autoddl_ref_chain_cost(Tp, L, K, s.data());
      sweeps[p * S + r] = nsweeps;
      for (int l = 0; l < L; ++l) strategy[(p * S + r) * L + l] = s[l];
    }
  }
  return 0;
}

// ---- R10 / PAPER.md:243 "records the best strategy": smallest cost over the starts, smallest start index on ties
extern "C" int autoddl_ref_best_of_starts(const int64_t* cost, int32_t Bp, int32_t S, int64_t* best_cost, int32_t* best_start) {
  if (!cost || !best_cost || !best_start || Bp < 1 || S < 1) return -1;
  for (int64_t p = 0; p < Bp; ++p) {
    int32_t arg = 0;
    for (int32_t s = 1; s < S; ++s)
      if (cost[p * S + s] < cost[p * S + arg]) arg = s;               // strict: the first start attaining the minimum
    best_cost[p] = cost[p * S + arg];
    best_start[p] = arg;
  }
  return 0;
}

// ---- R27: pipeline stages ("consecutive layers form a pipeline stage", 1F1B) -----------
// A stage is a contiguous segment [a, b) of the chain on its own sub-mesh; T / node / mask are the tables of the chain
// ON THAT SUB-MESH.  The first layer of a segment has no producer inside the stage (its input arrives from the previous
// stage by point-to-point transfer, already in the layout it needs), so only its node cost and penalty count:
//   f_a[j] = node[a][j] + PEN * [mask[a][j] == 0];  f_l[j] = min_i f_{l-1}[i] + T[l][i][j]  (a < l < b);
//   C(a, b) = min_j f_{b-1}[j]   -- the optimum of the segment over all K^(b-a) strategies.
// tri[a * (L + 1) + b] = C(a, b) for 0 <= a < b <= L, -1 elsewhere.
extern "C" int autoddl_ref_segment_optima(const int64_t* T, const int64_t* node, const uint8_t* mask, int32_t L, int32_t K,
                                          int64_t* tri) {
  if (!T || !node || !mask || !tri || L < 1 || K < 1) return -1;
  for (int64_t x = 0; x < (int64_t)L * (L + 1); ++x) tri[x] = -1;
  std::vector<int64_t> f(K), g(K);
  for (int32_t a = 0; a < L; ++a) {
    for (int j = 0; j < K; ++j) f[j] = node[(int64_t)a * K + j] + (mask[(int64_t)a * K + j] ? 0 : REF_PEN);
    for (int32_t b = a + 1; b <= L; ++b) {                           // segment [a, b): last layer b - 1
      if (b - 1 > a) {
        const int64_t* tile = T + (int64_t)(b - 1) * K * K;
        for (int j = 0; j < K; ++j) {
          int64_t best = f[0] + tile[j];
          for (int i = 1; i < K; ++i) {
            const int64_t v = f[i] + tile[(int64_t)i * K + j];
            if (v < best) best = v;
          }
          g[j] = best;
        }
        f.swap(g);
      }
      int64_t m = f[0];
      for (int j = 1; j < K; ++j) if (f[j] < m) m = f[j];
      tri[(int64_t)a * (L + 1) + b] = m;
    }
  }
  return 0;
}

// Point-to-point transfer at a stage boundary in front of layer b (a message of n bytes takes
// alpha + n beta; "point-to-point communications for transferring intermediate results between stages"):
// the input tensor of layer b, split evenly over the q devices of a stage, crosses the inter-node network once forward
// (activations) and once backward (their gradients) per micro-batch:
//   X(b) = 2 m (alpha_inter + ceil(in_rows_b in_cols_b act_bytes_b / q) beta_inter),   X(0) = 0.
extern "C" int autoddl_ref_stage_transfer(const ref_layer* layers, int32_t L, const ref_mesh* mesh, const ref_net* net,
                                          int64_t* xfer) {
  if (!layers || !mesh || !net || !xfer || L < 1) return -1;
  int64_t q = 1;
  for (int d = 0; d < mesh->ndim; ++d) q *= mesh->size[d];
  const int64_t m = net->micro_batches > 1 ? net->micro_batches : 1;
  xfer[0] = 0;
  for (int32_t b = 1; b < L; ++b) {
    const int64_t bytes = layers[b].in_rows * layers[b].in_cols * layers[b].act_bytes;
    xfer[b] = 2 * m * (net->alpha_ps[1] + ceil_div(bytes, q) * net->beta_ps_per_byte[1]);
  }
  return 0;
}

// Partition of the chain into `stages` contiguous non-empty segments.  Cost of a stage [a, b): its segment optimum plus
// the transfers at both of its boundaries, c(a, b) = C(a, b) + X(a) + [b < L] X(b).  objective 0: the SUM of the stage
// costs (total communication); objective 1: the MAX (the slowest stage sets the pace of a 1F1B pipeline).  Plain DP over
// the cuts: g_1[b] = c(0, b); g_k[b] = min_{a} comb(g_{k-1}[a], c(a, b)), smallest a on ties; cuts by back-tracking
// from g_stages[L].  cuts[0] = 0 < cuts[1] < ... < cuts[stages] = L.
extern "C" int autoddl_ref_pipeline_partition(const int64_t* tri, const int64_t* xfer, int32_t L, int32_t stages,
                                              int32_t objective, int64_t* value, int32_t* cuts) {
  if (!tri || !xfer || !value || !cuts || L < 1 || stages < 1 || stages > L || objective < 0 || objective > 1) return -1;
  const int64_t INF = INT64_MAX;
  std::vector<int64_t> g((size_t)(stages + 1) * (L + 1), INF);
  std::vector<int32_t> arg((size_t)(stages + 1) * (L + 1), -1);
  auto c = [&](int a, int b) { return tri[(int64_t)a * (L + 1) + b] + xfer[a] + (b < L ? xfer[b] : 0); };
  for (int b = 1; b <= L; ++b) { g[(size_t)1 * (L + 1) + b] = c(0, b); arg[(size_t)1 * (L + 1) + b] = 0; }
  for (int k = 2; k <= stages; ++k)
    for (int b = k; b <= L; ++b)
      for (int a = k - 1; a < b; ++a) {
        const int64_t prev = g[(size_t)(k - 1) * (L + 1) + a];
        if (prev == INF) continue;
        const int64_t cs = c(a, b);
        const int64_t v = objective == 0 ? prev + cs : (prev > cs ? prev : cs);
        if (v < g[(size_t)k * (L + 1) + b]) { g[(size_t)k * (L + 1) + b] = v; arg[(size_t)k * (L + 1) + b] = a; }
      }
  *value = g[(size_t)stages * (L + 1) + L];
  cuts[stages] = L;
  for (int k = stages; k >= 1; --k) cuts[k - 1] = arg[(size_t)k * (L + 1) + cuts[k]];
  return 0;
}

// Strategy of the whole chain under given cuts: every segment's optimum by the DP above with back-pointers (smallest
// index on ties, smallest end state), concatenated; seg_cost[k] = C(cuts[k], cuts[k+1]).
extern "C" int autoddl_ref_segment_strategies(const int64_t* T, const int64_t* node, const uint8_t* mask, int32_t L, int32_t K,
                                              const int32_t* cuts, int32_t stages, int64_t* seg_cost, int32_t* strategy) {
  if (!T || !node || !mask || !cuts || !seg_cost || !strategy || L < 1 || K < 1 || stages < 1) return -1;
  std::vector<int64_t> f(K), g(K);
  std::vector<int32_t> bp((size_t)L * K);
  for (int k = 0; k < stages; ++k) {
    const int a = cuts[k], b = cuts[k + 1];
    if (a < 0 || b > L || a >= b) return -1;
    for (int j = 0; j < K; ++j) f[j] = node[(int64_t)a * K + j] + (mask[(int64_t)a * K + j] ? 0 : REF_PEN);
    for (int l = a + 1; l < b; ++l) {
      const int64_t* tile = T + (int64_t)l * K * K;
      for (int j = 0; j < K; ++j) {
        int64_t best = f[0] + tile[j];
        int32_t ar = 0;
        for (int i = 1; i < K; ++i) {
          const int64_t v = f[i] + tile[(int64_t)i * K + j];
          if (v < best) { best = v; ar = i; }
        }
        g[j] = best;
        bp[(size_t)l * K + j] = ar;
      }
      f.swap(g);
    }
    int js = 0;
    for (int j = 1; j < K; ++j) if (f[j] < f[js]) js = j;
    seg_cost[k] = f[js];
    strategy[b - 1] = js;
    for (int l = b - 1; l > a; --l) strategy[l - 1] = bp[(size_t)l * K + strategy[l]];
  }
  return 0;
}

// ---- R19-R22: Metropolis-Hastings.  P(S) ~ exp(-beta Cost(S)), beta = 1 / tau; a proposal
// changes the signature of one layer; it is accepted with probability min(1, P(S_new) / P(S_old)).
extern "C" uint64_t autoddl_ref_rng(uint64_t seed, uint64_t n) {
  uint64_t z = seed + n * 0x9E3779B97F4A7C15ull;                    // splitmix64: state after n increments
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// -ln(x / 2^32) in Q16, x in [1, 2^32].  log2(x) = n + frac: n = index of the top bit; the 16 fraction bits come
// from squaring the mantissa m in [1, 2) sixteen times (m^2 >= 2 -> bit 1, halve), every product truncated to
// Q62.  Then -ln = (32 - log2 x) * ln 2 with ln 2 = 744261117 / 2^30 (truncated).
extern "C" int64_t autoddl_ref_neglog_q16(uint64_t x) {
  if (x < 1 || x > (1ull << 32)) return -1;
  int n = 0;
  while ((x >> (n + 1)) != 0) ++n;
  uint64_t m = x << (62 - n);                                        // Q62 in [2^62, 2^63)
  uint64_t frac = 0;
  for (int k = 0; k < 16; ++k) {
    const unsigned __int128 sq = (unsigned __int128)m * m;           // Q124
    m = (uint64_t)(sq >> 62);                                        // Q62 in [2^62, 2^64)
    frac <<= 1;
    if (m >= (1ull << 63)) { frac |= 1; m >>= 1; }
  }
  const int64_t log2_q16 = ((int64_t)n << 16) | (int64_t)frac;
  const int64_t nlog2_q16 = ((int64_t)32 << 16) - log2_q16;          // >= 0
  return (nlog2_q16 * 744261117ll) >> 30;
}

extern "C" int autoddl_ref_metropolis(const int64_t* T, int32_t Bp, int32_t L, int32_t K,
                                      const int32_t* init, int32_t S, int32_t nsteps, int64_t tau_ps, uint64_t seed,
                                      int64_t* best_cost, int32_t* best_strategy, int64_t* final_cost,
                                      int32_t* final_strategy, int32_t* accepted, int64_t* trace) {
  if (!T || !init || !best_cost || !best_strategy || !final_cost || !final_strategy || !accepted) return -1;
  if (Bp < 1 || L < 1 || K < 1 || S < 1 || nsteps < 0 || tau_ps < 0 || tau_ps >= ((int64_t)1 << 40)) return -1;
  std::vector<int32_t> s(L), sbest(L);
  for (int64_t p = 0; p < Bp; ++p) {
    const int64_t* Tp = T + p * L * K * K;
    for (int64_t r = 0; r < S; ++r) {
      const uint64_t chain = (uint64_t)(p * S + r);
      for (int l = 0; l < L; ++l) s[l] = init[(p * S + r) * L + l];
      int64_t cur = autoddl_ref_chain_cost(Tp, L, K, s.data());
      int64_t best = cur;
      sbest = s;
      int32_t nacc = 0;
      for (int64_t t = 0; t < nsteps; ++t) {
        const uint64_t base = ((chain << 32) + (uint64_t)t) * 4;
        const int32_t l = (int32_t)(autoddl_ref_rng(seed, base + 1) % (uint64_t)L);
        const int32_t c = (int32_t)(autoddl_ref_rng(seed, base + 2) % (uint64_t)K);
        const uint64_t x = (autoddl_ref_rng(seed, base + 3) >> 32) + 1;
        // Cost(S_new) - Cost(S_old): only the entries that touch layer l change
        const int32_t left = (l > 0) ? s[l - 1] : 0;
        int64_t d = Tp[((int64_t)l * K + left) * K + c] - Tp[((int64_t)l * K + left) * K + s[l]];
        if (l < L - 1)
          d += Tp[((int64_t)(l + 1) * K + c) * K + s[l + 1]] - Tp[((int64_t)(l + 1) * K + s[l]) * K + s[l + 1]];
        bool acc = d <= 0;
        if (!acc && d < ((int64_t)1 << 45)) acc = tau_ps * autoddl_ref_neglog_q16(x) >= (d << 16);
        if (acc) {
          s[l] = c;
          cur += d;
          ++nacc;
          if (cur < best) { best = cur; sbest = s; }
        }
        if (trace) trace[(p * S + r) * (int64_t)nsteps + t] = cur;
      }
      best_cost[p * S + r] = best;
      final_cost[p * S + r] = cur;
      accepted[p * S + r] = nacc;
      for (int l = 0; l < L; ++l) {
        best_strategy[(p * S + r) * L + l] = sbest[l];
        final_strategy[(p * S + r) * L + l] = s[l];
      }
    }
  }
  return 0;
}
