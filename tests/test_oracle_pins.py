"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test cites the passage of /root/reference/PAPER.md (quoted in tests/golden/*.txt or here)
or the invariant it checks.  None of them re-types the oracle's own loops: expected values are
hand arithmetic, the paper's printed numbers, closed forms, brute force, or numpy one-liners of
the textbook definition.
"""
import itertools

import numpy as np
import pytest

from oracle import ref
from paper_2301_06813_b200 import configs as cf
from tests.conftest import read_golden

S0, S1, B, P = 0, 1, 2, 3
PEN = 1 << 50


@pytest.fixture(scope="module")
def cfg1():
    w = cf.config1_tiny()
    T, node, mask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    return w, T, node, mask


# ---- P1: Table 2 hand values --------------------------------------------------
def test_table2_hand_values():
    g = read_golden("table2_hand_values.txt")
    a = (2**20, 4, 5_000_000, 3)
    b = (1_000_001, 8, 20_000_000, 40)
    for tag, args in (("A", a), ("B", b)):
        assert ref.collective(ref.AG, *args) == g[f"{tag}_allgather"]
        assert ref.collective(ref.RS, *args) == g[f"{tag}_reducescatter"]
        assert ref.collective(ref.AR, *args) == g[f"{tag}_allreduce"]
        assert ref.collective(ref.A2A, *args) == g[f"{tag}_alltoall"]


# ---- P2: identities between the rows of Table 2 ----------------------------------------------------
@pytest.mark.parametrize("n", [1, 7, 4096, 1_000_001, 3 * 2**33])
@pytest.mark.parametrize("p", [1, 2, 3, 8, 16, 64])
def test_table2_identities(n, p):
    al, be = 20_000_000, 40
    ag, rs = ref.collective(ref.AG, n, p, al, be), ref.collective(ref.RS, n, p, al, be)
    ar, a2a = ref.collective(ref.AR, n, p, al, be), ref.collective(ref.A2A, n, p, al, be)
    assert ag == rs                                     # one row of Table 2
    if p == 1:
        assert ag == ar == a2a == 0                     # a group of one does not communicate
        return
    # north_star: "all-reduce cost equals reduce-scatter plus all-gather"; Table 2 prints (2p-1) alpha
    # for AllReduce, one alpha more than 2(p-1) (R3/A4): equal up to that alpha, exactly with alpha=0
    assert ar - al == rs + ag
    assert ref.collective(ref.AR, n, p, 0, be) == 2 * ref.collective(ref.AG, n, p, 0, be)
    assert ref.collective(ref.AG, n, p, al, 0) == (p - 1) * al     # latency term alone
    assert ref.collective(ref.A2A, n, p, 0, be) == n * be          # AlltoAll beta term is n*beta as printed
    if n % p == 0:                                      # exact (p-1)/p * n * beta when p divides n
        assert ref.collective(ref.AG, n, p, 0, be) * p == (p - 1) * n * be


# ---- P3: the paper's worked number, 3.75 billion elements = 15 GB -------------------
def test_paper_attention_15GB():
    g = read_golden("paper_attention_15GB.txt")
    mesh = ref.make_mesh((4, 16), (cf.INTER, cf.INTER))
    net = ref.make_net((0, 0), (1, 1))                  # cost == bytes on the wire
    rows, cols, eb = 2**20, 8192, 4
    fwd = ref.reshard(rows, cols, eb, (S0, S1), (S0, B), mesh, net)
    bwd = ref.reshard(rows, cols, eb, (S0, P), (S0, S1), mesh, net)   # dual(b) -> dual(a)
    assert fwd == g["fwd_allgather_bytes"]
    assert bwd == g["bwd_reducescatter_bytes"]
    assert fwd + bwd == g["total_bytes"] == 15 * 2**30
    assert (fwd + bwd) // eb == g["total_elements"]
    # the same through the edge cost: a GEMM producing (S0,S1) [sigs 0,1] feeding one that wants (S0,B) [sigs 0,1->I=(S0,B)]
    prev = cf.gemm(rows, cols, cols, 4, 4, 8)
    cur = cf.gemm(rows, cols, cols, 4, 4, 8)
    assert ref.edge_cost(prev, cur, 0 * 6 + 1, 0 * 6 + 1, mesh, net) == g["total_bytes"]


# ---- hand cells of config 1 and P4: data parallel closed form -----------------
def test_hand_cells_config1(cfg1):
    g = read_golden("hand_cells.txt")
    w, T, node, mask = cfg1
    assert T[0, 1, 14, 7] == g["T_1_14_7"]
    assert node[0, 1, 7] == 0
    for l in range(4):
        assert node[0, l, 0] == g["V_sig0"]
        assert T[0, l, 0, 0] == g["V_sig0"]             # sig 0 -> sig 0: no redistribution at all
    assert ref.chain_cost(T[0], [0, 0, 0, 0]) == g["cost_all_sig0"]
    assert mask.all()                                   # no cap, splits within limits


def test_data_parallel_has_no_redistribution():
    """with p1 = p2 = 1 the SBP matmul is data parallelism: the only communication is
    the all-reduce of W's gradient."""
    for k in (2, 3):
        w = cf.CONFIGS[k]()
        mesh, net = ref.mesh_of(w), ref.net_of(w)
        lay = w.layers[0]
        for l in range(1, min(w.L, 10)):
            assert ref.edge_cost(lay[l - 1], lay[l], 0, 0, mesh, net) == 0


# ---- P5: 3D SBP matmul keeps n^2/p^(2/3) per device ---------------------------------
@pytest.mark.parametrize("q,n", [(2, 64), (4, 1024), (8, 12288)])
def test_3d_matmul_local_sizes(q, n):
    mesh = ref.make_mesh((q, q, q), (cf.INTER, cf.INTER, cf.INTRA))
    sig = 0 * 36 + 1 * 6 + 2                            # levels use signatures (0, 1, 2): PAPER.md:193
    v, I, W, O = ref.sig_states(cf.GEMM, sig, mesh)
    assert v == 1
    assert I == (S0, B, S1) and W == (B, S1, S0) and O == (S0, S1, P)      # verbatim PAPER.md:193
    want = n * n // (q * q)                             # n^2 / p^(2/3), p = q^3
    assert ref.local_size(n, n, I, mesh) == want
    assert ref.local_size(n, n, W, mesh) == want
    assert ref.local_size(n, n, O, mesh) == want
    assert ref.layer_mem(cf.gemm(n, n, n, 2, 4, 18), sig, mesh) == want * 18 + 2 * want * 2


def test_local_size_ceil():
    mesh = ref.make_mesh((4, 8), (1, 0))
    assert ref.local_size(1001, 777, (S0, S1), mesh) == 251 * 98
    assert ref.local_size(1001, 777, (S0, S0), mesh) == 32 * 777
    assert ref.local_size(1001, 777, (B, P), mesh) == 1001 * 777


# ---- P6: link class of a collective is the level's ----------------------------------
def test_link_rule_paper_example():
    """on 2 nodes x 4 GPUs, (S0:(1,2), B:(2,2)) -> B:(2,4) "only intra-node
    communication is required"; (S0:(2,1), B:(1,4)) -> B:(2,4) "inter-node communication is required"."""
    net = ref.make_net((1, 1000), (0, 0))               # cost = (p-1) * alpha of the link used
    mesh = ref.make_mesh((2, 2, 2), (cf.INTER, cf.INTRA, cf.INTRA))
    assert ref.reshard(64, 64, 4, (B, S0, B), (B, B, B), mesh, net) == 1          # intra alpha only
    assert ref.reshard(64, 64, 4, (S0, B, B), (B, B, B), mesh, net) == 1000       # inter alpha only


# ---- P7: identity costs nothing; forward == backward when every split divides ----------------------
def _all_states(D):
    return list(itertools.product(range(4), repeat=D))


@pytest.mark.parametrize("sizes,links", [((2, 2), (1, 0)), ((4, 8), (1, 0)), ((2, 3, 4), (1, 1, 0))])
def test_reshard_identity_and_symmetry(sizes, links):
    mesh = ref.make_mesh(sizes, links)
    net = ref.make_net(cf.ALPHA_PS, (3, 40))
    dual = {S0: S0, S1: S1, B: P, P: B}
    rows, cols = 2**6 * 3**3, 2**7 * 3**2                 # divisible by every product of sizes
    for a in _all_states(len(sizes)):
        assert ref.reshard(rows, cols, 2, a, a, mesh, net) == 0
        for b in _all_states(len(sizes)):
            f = ref.reshard(rows, cols, 2, a, b, mesh, net)
            assert f >= 0
            bw = ref.reshard(rows, cols, 2, tuple(dual[x] for x in b), tuple(dual[x] for x in a), mesh, net)
            assert f == bw, (a, b)


def test_reshard_free_moves():
    """B->S (slice), S->P and B->P (zero fill) move no data."""
    mesh = ref.make_mesh((4, 4), (1, 0))
    net = ref.make_net(cf.ALPHA_PS, (3, 40))
    for a, b in [((B, B), (S0, S1)), ((S0, S1), (P, P)), ((B, B), (P, P)), ((B, S0), (S1, P))]:
        assert ref.reshard(4096, 4096, 2, a, b, mesh, net) == 0


def test_edge_layer0_and_invalid(cfg1):
    w, T, node, mask = cfg1
    # R8: layer 0 has no producer: every row of tile 0 is the same
    assert (T[0, 0] == T[0, 0, 0][None, :]).all()
    # ATTN: signatures using a P state are invalid: PEN on the column, zero edge on the row
    w3 = cf.config3_transformer24()
    T3, node3, mask3 = ref.build_tables(w3.layers[:, :3], ref.mesh_of(w3), ref.net_of(w3))
    for j in range(36):
        valid = all(d in (0, 1, 3) for d in divmod(j, 6))
        if not valid:
            assert mask3[0, 1, j] == 0 and node3[0, 1, j] == 0
            assert (T3[0, 1, :, j] == PEN).all()
            assert (T3[0, 2, j, :] == node3[0, 2][None, :] + np.where(mask3[0, 2] == 1, 0, PEN)).all()


# ---- P8: DP optimum == exhaustive search --------------------------------------------
def test_dp_equals_brute_force_config1(cfg1):
    g = read_golden("survey_crosscheck.txt")
    w, T, _, _ = cfg1
    bc, bs = ref.brute_force(T[0])                      # 36^4 = 1,679,616 strategies
    dc, ds = ref.chain_dp(T)
    assert bc == dc[0] == g["config1_dp"]
    assert ref.chain_cost(T[0], ds[0]) == dc[0]
    assert ref.chain_cost(T[0], bs) == bc


def _random_tables(rng, Bp, L, K, ties=True):
    hi = 12 if ties else 10**9                          # small range -> many exact ties
    T = rng.integers(0, hi, size=(Bp, L, K, K)).astype(np.int64)
    T[rng.random(T.shape) < 0.1] += PEN
    return T


@pytest.mark.parametrize("L,K", [(1, 6), (2, 6), (5, 6), (8, 6), (3, 36), (6, 4)])
def test_dp_equals_brute_force_random(L, K):
    rng = np.random.default_rng(100 * L + K)
    T = _random_tables(rng, 6, L, K, ties=(L % 2 == 1))
    dc, ds = ref.chain_dp(T)
    for p in range(T.shape[0]):
        bc, bs = ref.brute_force(T[p])
        assert bc == dc[p]
        assert ref.chain_cost(T[p], ds[p]) == dc[p]
        # independent python enumeration of the definition Cost(S) = sum_l T[l][s_{l-1}][s_l], s_{-1}=0
        if K ** L <= 50_000:
            best = min(sum(int(T[p, l, (s[l - 1] if l else 0), s[l]]) for l in range(L))
                       for s in itertools.product(range(K), repeat=L))
            assert best == bc


def test_dp_tie_break_is_lowest_index():
    """all-equal tables: every strategy is optimal; the procedure must return all zeros"""
    T = np.full((1, 5, 6, 6), 7, np.int64)
    c, s = ref.chain_dp(T)
    assert c[0] == 35 and s[0].tolist() == [0] * 5
    # unique optimum planted on high indices must still be found
    T = np.full((1, 4, 6, 6), 9, np.int64)
    path = [5, 3, 4, 2]
    prev = 0
    for l, j in enumerate(path):
        T[0, l, prev, j] = 1
        prev = j
    c, s = ref.chain_dp(T)
    assert c[0] == 4 and s[0].tolist() == path


def test_dp_matches_survey_crosscheck():
    g = read_golden("survey_crosscheck.txt")
    for k, key in ((2, "config2_dp"), (3, "config3_dp")):
        w = cf.CONFIGS[k]()
        T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
        c, s = ref.chain_dp(T)
        assert c[0] == g[key]
        assert ref.chain_cost(T[0], s[0]) == c[0]
    w = cf.config4_batched(Bp=1)
    assert int(w.layers["M"][0, 0]) == 616 and w.layers["Kd"][0, :5].tolist() == [404, 552, 4160, 928, 392]
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    assert ref.chain_dp(T)[0][0] == g["config4_problem0_dp"]


def test_vgg_strategy_shape():
    """convolutions use pure data parallelism (S0:p); the dense layers' weights are not replicated."""
    w = cf.config2_vgg16()
    mesh = ref.mesh_of(w)
    T, _, _ = ref.build_tables(w.layers, mesh, ref.net_of(w))
    _, s = ref.chain_dp(T)
    for l in range(12):
        v, I, W, O = ref.sig_states(cf.GEMM, int(s[0, l]), mesh)
        assert I[0] == S0 and O[0] == S0
    for l in (13, 14, 15):
        v, I, W, O = ref.sig_states(cf.GEMM, int(s[0, l]), mesh)
        assert W[0] != B


# ---- P9: Coordinate Descent properties ------------------------------------------
def _check_cd(T, init, max_sweeps=64):
    cost, strat, sweeps, trace = ref.coord_descent(T, init, max_sweeps, want_trace=True)
    dpc, _ = ref.chain_dp(T)
    Bp, L, K, _ = T.shape
    for p in range(Bp):
        for r in range(init.shape[1]):
            s = strat[p, r]
            # returned cost is Cost(s) by the definition
            prev = 0; tot = 0
            for l in range(L):
                tot += int(T[p, l, prev, s[l]]); prev = int(s[l])
            assert tot == cost[p, r]
            assert dpc[p] <= cost[p, r]                 # the optimum is never above a CD result
            n = sweeps[p, r]
            assert 1 <= n <= max_sweeps
            # "guarantees monotonic cost reduction": per update, never up
            tr = trace[p, r, :n].reshape(-1)
            start_cost = ref.chain_cost(T[p], init[p, r])
            seq = np.concatenate([[start_cost], tr])
            assert (np.diff(seq) <= 0).all()
            assert tr[-1] == cost[p, r]
            if n < max_sweeps:
                # fixed point: every s_l is the LOWEST-index minimiser given its neighbours (1-opt)
                for l in range(L):
                    left = s[l - 1] if l else 0
                    g = T[p, l, left, :].copy()
                    if l < L - 1:
                        g = g + T[p, l + 1, :, s[l + 1]]
                    assert int(np.argmin(g)) == s[l]    # numpy argmin returns the first minimum
                # the last sweep changed nothing: its trace is flat
                assert (trace[p, r, n - 1] == cost[p, r]).all()
    return cost, strat, sweeps


def test_cd_properties_random():
    rng = np.random.default_rng(7)
    for (L, K) in [(1, 6), (2, 6), (9, 6), (7, 36)]:
        T = _random_tables(rng, 4, L, K, ties=True)
        init = rng.integers(0, K, size=(4, 5, L)).astype(np.int32)
        _check_cd(T, init)


def test_cd_properties_configs():
    for k in (1, 2, 3):
        w = cf.CONFIGS[k]()
        T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
        init = w.cd_init()[:, :24]
        _check_cd(T, init, w.max_sweeps)


def test_cd_fixed_point_start_and_sweep_cap():
    rng = np.random.default_rng(11)
    T = _random_tables(rng, 3, 8, 6, ties=False)
    init = rng.integers(0, 6, size=(3, 4, 8)).astype(np.int32)
    cost, strat, sweeps = ref.coord_descent(T, init)
    c2, s2, n2 = ref.coord_descent(T, strat)            # restart from the fixed points
    assert (n2 == 1).all() and (s2 == strat).all() and (c2 == cost).all()
    c1, s1, n1 = ref.coord_descent(T, init, max_sweeps=1)
    assert (n1 == 1).all()
    # DP optimum is itself a fixed point in cost: CD started there cannot go below it
    dc, ds = ref.chain_dp(T)
    c3, _, _ = ref.coord_descent(T, ds[:, None, :].copy())
    assert (c3[:, 0] == dc).all()


def test_cd_first_update_by_hand():
    """Gauss-Seidel order: the update of layer 1 must see the NEW s_0."""
    K = 6
    T = np.full((1, 2, K, K), 100, np.int64)
    T[0, 0, 0, :] = [5, 4, 3, 2, 1, 9]                  # layer 0 alone prefers c = 4
    T[0, 1, :, :] = 50
    T[0, 1, 4, 2] = 0                                   # given s_0 = 4, layer 1 wants 2
    T[0, 1, 0, 3] = 0                                   # given the OLD s_0 = 0 it would want 3
    T[0, 1, 0, 0] = 48                                  # make start [0,0]: g_0(c) = T0[0][c] + T1[c][0]
    cost, strat, sweeps = ref.coord_descent(T, np.zeros((1, 1, 2), np.int32))
    assert strat[0, 0].tolist() == [4, 2] and cost[0, 0] == 1 and sweeps[0, 0] == 2


# ---- P10: penalty bookkeeping ------------------------------------------------------------------
def test_penalty_counts_infeasible_layers():
    w = cf.config3_transformer24()
    T, node, mask = ref.build_tables(w.layers[:, :10], ref.mesh_of(w), ref.net_of(w))
    rng = np.random.default_rng(3)
    for _ in range(50):
        s = rng.integers(0, 36, size=10)
        c = ref.chain_cost(T[0], s)
        bad = sum(1 for l in range(10) if mask[0, l, s[l]] == 0)
        assert c >> 50 == bad
        assert (c < PEN) == (bad == 0)


def test_memory_mask_hand_value():
    """PARITY UNPINNED against the paper (no formula printed); this only fixes our own
    definition at a hand-computed point: VGG FC1 (64 x 25088 x 4096, fp32, 12 B/weight), 8 x 1 mesh, cap 16e9/16."""
    w = cf.config2_vgg16()
    mesh, net = ref.mesh_of(w), ref.net_of(w)
    fc1 = w.layers[0, 13]
    # sig (0,*) : W replicated: 25088*4096*12 + (8*25088 + 8*4096)*4 = 1,233,125,376 + 933,888 > 1e9
    assert ref.layer_mem(fc1, 0, mesh) == 25088 * 4096 * 12 + (8 * 25088 + 8 * 4096) * 4
    assert ref.feasible(fc1, 0, 16, mesh, net) == 0
    # sig (1,*) : W split on columns over 8 nodes: 25088*512*12 + (64*25088 + 64*512)*4
    assert ref.layer_mem(fc1, 6, mesh) == 25088 * 512 * 12 + (64 * 25088 + 64 * 512) * 4
    assert ref.feasible(fc1, 6, 16, mesh, net) == 1
    # split limit: batch 64 cannot be split 4*8 = 32 > 8 ways for config 3's attention rows
    w3 = cf.config3_transformer24()
    at = w3.layers[0, 1]
    assert ref.feasible(at, 0 * 6 + 0, 120, ref.mesh_of(w3), ref.net_of(w3)) == 0     # rows split 32 > 8
    assert ref.feasible(at, 0 * 6 + 1, 120, ref.mesh_of(w3), ref.net_of(w3)) == 1     # rows 4, heads 8


def test_splitmix64_known_answer():
    r = cf.SplitMix64(0)
    assert r.next() == 0xE220A8397B1DCDAF               # published splitmix64 test vector, seed 0
    a = cf.SplitMix64(5); b = cf.SplitMix64(5)
    assert [a.next() for _ in range(9)] == b.next_array(9).tolist()
