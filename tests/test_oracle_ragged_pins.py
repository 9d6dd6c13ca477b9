"""Pins of the CPU oracle where dimensions are NOT divisible by the splits and element sizes differ between
neighbouring layers (no GPU).  Expected values are the hand arithmetic of tests/golden/ragged_hand_cells.txt
(PAPER.md:197-199 path, Table 2, readings DESIGN.md R2-R7), never an output of the oracle.

What each pin fixes (a one-line mistake of that kind fails it; tests/test_oracle_mutations.py replays them):
  level order and message size of the all-to-all phase        test_alltoall_both_levels_ragged
  scatter axis of P -> B, order of the reduce / gather phases test_reduce_and_gather_ragged
  the paper's own path on three levels                        test_paper_path_three_levels_ragged
  forward leg != backward leg, and E = fwd + bwd              test_edge_forward_differs_from_backward
  whose element size and whose tensor prices an edge          test_edge_uses_consumer_tensor_and_element_size
  weight-gradient all-reduce of the LOCAL weight              test_node_cost_local_weight_ragged
  boundaries of the split limits and of the memory cap        test_feasible_boundaries
  first strategy attaining the best cost in Metropolis        test_metropolis_best_is_first_attained
"""
import numpy as np

from oracle import ref
from paper_2301_06813_b200 import configs as cf
from tests.conftest import read_golden

S0, S1, B, P = 0, 1, 2, 3
PEN = 1 << 50
G = read_golden("ragged_hand_cells.txt")

MESH_A = ((4, 8), (cf.INTER, cf.INTRA))
ROWS, COLS = 1001, 777


def _mesh_a():
    return ref.make_mesh(*MESH_A)


def _net():
    return ref.make_net(cf.ALPHA_PS, (3, 40))


def test_alltoall_both_levels_ragged():
    mesh, net = _mesh_a(), _net()
    assert ref.reshard(ROWS, COLS, 2, (S0, S0), (S1, S1), mesh, net) == G["a2a_S0S0_to_S1S1_eb2"]
    assert ref.reshard(ROWS, COLS, 2, (S1, S1), (S0, S0), mesh, net) == G["a2a_S1S1_to_S0S0_eb2"]
    assert G["a2a_S0S0_to_S1S1_eb2"] != G["a2a_S1S1_to_S0S0_eb2"]


def test_reduce_and_gather_ragged():
    mesh, net = _mesh_a(), _net()
    assert ref.reshard(ROWS, COLS, 2, (P, P), (B, B), mesh, net) == G["rs_ag_PP_to_BB_eb2"]
    assert ref.reshard(ROWS, COLS, 2, (P, S0), (S1, B), mesh, net) == G["rs_then_ag_PS0_to_S1B_eb2"]
    assert ref.reshard(ROWS, COLS, 2, (S0, S1), (B, B), mesh, net) == G["ag_S0S1_to_BB_eb2"]
    assert ref.reshard(ROWS, COLS, 2, (P, P), (S0, S1), mesh, net) == G["rs_PP_to_S0S1_eb2"]


def test_paper_path_three_levels_ragged():
    """(S0:p0, S1:p1, P:p2) -> (S0:p0, S1:p1*p2) -> (S0:p0', B:p1', S1:p2') is a ReduceScatter then an
    AllGather 'in both the forward path and the backward path'."""
    mesh = ref.make_mesh((2, 3, 5), (cf.INTER, cf.INTER, cf.INTRA))
    net = _net()
    fwd = ref.reshard(ROWS, COLS, 4, (S0, S1, P), (S0, B, S1), mesh, net)
    assert fwd == G["paper_path_S0S1P_to_S0BS1_eb4"]
    # backward: dual(b) -> dual(a) = (S0,P,S1) -> (S0,S1,B): reduce-scatter over level 1, all-gather over level 2: the
    # same two collectives on the same two local tensors
    assert ref.reshard(ROWS, COLS, 4, (S0, P, S1), (S0, S1, B), mesh, net) == fwd
    # through the table: producer signature (0,1,2) has O = (S0,S1,P), consumer signature (0,3,2) has I = (S0,B,S1)
    prev = cf.gemm(ROWS, 640, COLS, 4, 4, 8)
    cur = cf.gemm(ROWS, COLS, 512, 4, 4, 8)
    assert ref.sig_states(cf.GEMM, 0 * 36 + 1 * 6 + 2, mesh)[3] == (S0, S1, P)
    assert ref.sig_states(cf.GEMM, 0 * 36 + 3 * 6 + 2, mesh)[1] == (S0, B, S1)
    assert ref.edge_cost(prev, cur, 0 * 36 + 1 * 6 + 2, 0 * 36 + 3 * 6 + 2, mesh, net) == 2 * fwd


def test_edge_forward_differs_from_backward():
    mesh, net = _mesh_a(), _net()
    prev = cf.gemm(ROWS, 640, COLS, 2, 4, 18)
    cur = cf.gemm(ROWS, COLS, 512, 2, 4, 18)
    # signature (0,0) = index 0: O = (S0,S0); signature (2,2) = index 14: I = (S1,S1)
    assert ref.sig_states(cf.GEMM, 0, mesh)[3] == (S0, S0) and ref.sig_states(cf.GEMM, 14, mesh)[1] == (S1, S1)
    e = ref.edge_cost(prev, cur, 0, 14, mesh, net)
    assert e == G["edge_0_14_consumer_eb2"] == G["a2a_S0S0_to_S1S1_eb2"] + G["a2a_S1S1_to_S0S0_eb2"]
    assert e != 2 * G["a2a_S0S0_to_S1S1_eb2"] and e != 2 * G["a2a_S1S1_to_S0S0_eb2"]
    # and in the table itself (layer 1, row 0, column 14), on top of the node cost of the column
    layers = np.stack([prev, cur]).reshape(1, 2)
    T, node, mask = ref.build_tables(layers, mesh, net)
    assert T[0, 1, 0, 14] == e + node[0, 1, 14] and mask[0, 1, 14] == 1


def test_edge_uses_consumer_tensor_and_element_size():
    """R5: the redistributed tensor is the consumer's input (in_rows x in_cols, act_bytes of the consumer)."""
    mesh, net = _mesh_a(), _net()
    for prev_eb, cur_eb, key in ((4, 2, "edge_0_14_consumer_eb2"), (2, 4, "edge_0_14_consumer_eb4"),
                                 (2, 2, "edge_0_14_consumer_eb2"), (4, 4, "edge_0_14_consumer_eb4")):
        # the producer's own M x N (333 x 4096) is NOT the tensor that moves
        prev = cf.gemm(333, 640, 4096, prev_eb, 4, 18)
        cur = cf.gemm(555, COLS, 512, cur_eb, 4, 18, in_rows=ROWS, in_cols=COLS)
        assert ref.edge_cost(prev, cur, 0, 14, mesh, net) == G[key]
        T, node, _ = ref.build_tables(np.stack([prev, cur]).reshape(1, 2), mesh, net)
        assert T[0, 1, 0, 14] - node[0, 1, 14] == G[key]


def test_node_cost_local_weight_ragged():
    mesh, net = _mesh_a(), _net()
    lay = cf.gemm(64, 777, 1001, 2, 4, 18)
    assert ref.sig_states(cf.GEMM, 6, mesh)[2] == (S1, B) and ref.sig_states(cf.GEMM, 15, mesh)[2] == (S0, B)
    assert ref.node_cost(lay, 6, mesh, net) == G["node_sig6_ragged"]
    assert ref.node_cost(lay, 15, mesh, net) == G["node_sig15_ragged"]
    assert ref.sig_states(cf.GEMM, 30, mesh)[2] == (P, B) and ref.sig_states(cf.GEMM, 35, mesh)[2] == (P, P)
    assert ref.node_cost(lay, 30, mesh, net) == G["node_sig30_ragged"]
    assert ref.node_cost(lay, 35, mesh, net) == G["node_sig35_ragged"] == 0
    T, node, _ = ref.build_tables(np.stack([lay]).reshape(1, 1), mesh, net)
    assert node[0, 0, 6] == G["node_sig6_ragged"] and T[0, 0, 0, 6] == G["node_sig6_ragged"]
    assert node[0, 0, 15] == G["node_sig15_ragged"] and T[0, 0, 3, 15] == G["node_sig15_ragged"]


def test_feasible_boundaries():
    """R7 (ours; the paper prints no formula): split <= limit and mem <= floor(cap / L), both inclusive."""
    mesh = _mesh_a()
    L = 3
    lay = cf.gemm(1001, 777, 500, 2, 4, 18)
    mem = G["mem_sig1_ragged"]
    assert ref.layer_mem(lay, 1, mesh) == mem
    for cap, want in ((L * mem, 1), (L * mem + 2, 1), (L * mem - 1, 0), (0, 1)):
        net = ref.make_net(cf.ALPHA_PS, (3, 40), mem_cap_bytes=cap)
        assert ref.feasible(lay, 1, L, mesh, net) == want, cap
        T, _, mask = ref.build_tables(np.stack([lay] * L).reshape(1, L), mesh, net)
        assert mask[0, 0, 1] == want and (T[0, 0, 0, 1] >= PEN) == (want == 0)
    net = _net()
    # signature (1,1) = index 7: O = (S1,S1): column split 32; signature (0,0): row split 32; (0,1): rows 4, columns 8
    for sig, rows_lim, cols_lim, want in ((7, 1, 32, 1), (7, 1, 31, 0), (7, 1, 33, 1), (0, 32, 1, 1), (0, 31, 1, 0),
                                          (1, 4, 8, 1), (1, 3, 8, 0), (1, 4, 7, 0)):
        lay = cf.gemm(1001, 777, 500, 2, 4, 18, max_rows=rows_lim, max_cols=cols_lim)
        assert ref.feasible(lay, sig, L, mesh, net) == want, (sig, rows_lim, cols_lim)


def test_metropolis_best_is_first_attained():
    """R22: the best strategy is the FIRST one attaining the smallest cost.  On an all-equal table every proposal is
    accepted (dC = 0) and no cost is ever smaller than the start's: best = the start, final = somewhere else."""
    L, K = 5, 6
    T = np.full((1, L, K, K), 11, np.int64)
    init = np.array([[[3, 1, 4, 1, 5]]], np.int32)
    bc, bs, fc, fs, acc = ref.metropolis(T, init, 200, 1_000_000, seed=3)
    assert bc[0, 0] == fc[0, 0] == 11 * L and acc[0, 0] == 200
    assert bs[0, 0].tolist() == init[0, 0].tolist()
    assert fs[0, 0].tolist() != init[0, 0].tolist()
    # a planted strictly better strategy reached later replaces it, and only the first visit counts
    T2 = T.copy()
    T2[0, 0, 0, 2] = 1                                   # every strategy with s_0 = 2 costs 10 less, all tie among them
    bc, bs, fc, fs, acc, tr = ref.metropolis(T2, init, 400, 1_000_000_000, seed=3, want_trace=True)
    first = int(np.argmax(tr[0, 0] == bc[0, 0]))
    assert bc[0, 0] == 11 * L - 10 and tr[0, 0, first] == bc[0, 0] and (tr[0, 0, :first] > bc[0, 0]).all()
    assert bs[0, 0, 0] == 2
    # replay the draws up to the first visit: the recorded best strategy is the state right after step `first`
    s = init[0, 0].tolist()
    cur = 11 * L
    for t in range(first + 1):
        base = 4 * t                                    # chain 0
        l = ref.rng(3, base + 1) % L
        c = ref.rng(3, base + 2) % K
        s2 = list(s); s2[l] = c
        c2 = sum(int(T2[0, k, (s2[k - 1] if k else 0), s2[k]]) for k in range(L))
        if c2 == cur or tr[0, 0, t] == c2:              # dC = 0 is always accepted; otherwise the traced cost tells
            s, cur = s2, c2
    assert cur == bc[0, 0] and bs[0, 0].tolist() == s
