"""Pins of the oracle's pipeline-stage enumeration (R27), no GPU.

What is fixed by mathematics: a segment optimum is the minimum over all K^(b-a) strategies of the segment (brute force),
one stage is the whole-chain DP, the partition value is the minimum over all cut sets (brute force over combinations).
What is OURS (the paper prints no stage-cost model): the transfer term and the sum / max objective -- pinned only at
hand-computed points of our own definition (tests/golden/pipeline_hand_values.txt)."""
import itertools

import numpy as np
import pytest

from oracle import ref
from paper_2301_06813_b200 import configs as cf
from tests.conftest import read_golden

PEN = 1 << 50
G = read_golden("pipeline_hand_values.txt")


def _tables(w):
    T, node, mask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    return T[0], node[0], mask[0]


def _random_problem(rng, L, K, hi=50):
    T = rng.integers(0, hi, size=(L, K, K)).astype(np.int64)
    node = rng.integers(0, hi, size=(L, K)).astype(np.int64)
    mask = (rng.random((L, K)) > 0.15).astype(np.uint8)
    T += node[:, None, :] + np.where(mask == 1, 0, PEN)[:, None, :]
    return T, node, mask


def _segment_as_chain(T, node, mask, a, b):
    """the segment [a, b) as a chain of its own: every row of its first tile is node + penalty (no producer)"""
    sub = T[a:b].copy()
    sub[0] = (node[a] + np.where(mask[a] == 1, 0, PEN))[None, :]
    return sub


@pytest.mark.parametrize("k", [1, 2, 3])
def test_one_stage_is_the_chain_dp(k):
    w = cf.CONFIGS[k]()
    T, node, mask = _tables(w)
    tri = ref.segment_optima(T, node, mask)
    dc, ds = ref.chain_dp(T[None])
    assert tri[0, w.L] == dc[0]
    # and every prefix [0, b) is the DP of the truncated chain
    for b in (1, 2, w.L // 2):
        assert tri[0, b] == ref.chain_dp(T[None, :b])[0][0]
    assert (tri[np.tril_indices(w.L, 0, w.L + 1)] == -1).all()      # a >= b: not a segment


@pytest.mark.parametrize("L,K", [(1, 6), (4, 6), (5, 6), (3, 36)])
def test_segment_optima_equal_brute_force(L, K):
    rng = np.random.default_rng(10 * L + K)
    T, node, mask = _random_problem(rng, L, K, hi=9 if L % 2 else 10**6)
    tri = ref.segment_optima(T, node, mask)
    for a in range(L):
        for b in range(a + 1, L + 1):
            bc, _ = ref.brute_force(_segment_as_chain(T, node, mask, a, b))
            assert tri[a, b] == bc, (a, b)
        assert (np.diff(tri[a, a + 1:]) >= 0).all()                 # costs are non-negative: longer segments cost more


def test_segment_first_layer_has_no_edge():
    """a segment that starts at layer a > 0 pays node + penalty there, NOT the redistribution from layer a - 1"""
    w = cf.config1_tiny()
    T, node, mask = _tables(w)
    tri = ref.segment_optima(T, node, mask)
    for a in range(w.L):
        assert tri[a, a + 1] == (node[a] + np.where(mask[a] == 1, 0, PEN)).min()
    assert tri[1, 2] == 0                                           # some signature keeps W un-replicated: no communication


def _evaluate(tri, xfer, cuts, objective):
    L = tri.shape[0]
    costs = [int(tri[a, b]) + int(xfer[a]) + (int(xfer[b]) if b < L else 0) for a, b in zip(cuts[:-1], cuts[1:])]
    return sum(costs) if objective == 0 else max(costs)


@pytest.mark.parametrize("L", [1, 2, 5, 8])
def test_partition_equals_brute_force_over_cut_sets(L):
    rng = np.random.default_rng(L)
    T, node, mask = _random_problem(rng, L, 6, hi=40)
    tri = ref.segment_optima(T, node, mask)
    xfer = np.concatenate([[0], rng.integers(0, 60, L - 1)]).astype(np.int64)
    for stages in range(1, min(L, 4) + 1):
        for objective in (0, 1):
            val, cuts = ref.pipeline_partition(tri, xfer, stages, objective)
            best = min(_evaluate(tri, xfer, (0,) + c + (L,), objective) for c in itertools.combinations(range(1, L), stages - 1))
            assert val == best, (stages, objective)
            assert cuts[0] == 0 and cuts[-1] == L and (np.diff(cuts) >= 1).all() and len(cuts) == stages + 1
            assert _evaluate(tri, xfer, cuts.tolist(), objective) == val
    # one stage: the whole chain, no transfer
    val, cuts = ref.pipeline_partition(tri, xfer, 1, 1)
    assert val == tri[0, L] and cuts.tolist() == [0, L]


def test_partition_toy_by_hand():
    """three layers, two stages: the arithmetic is written out in tests/golden/pipeline_hand_values.txt"""
    L = 3
    tri = np.full((L, L + 1), -1, np.int64)
    tri[0, 1], tri[0, 2], tri[0, 3], tri[1, 2], tri[1, 3], tri[2, 3] = 5, 7, 16, 1, 4, 2
    xfer = np.array([0, 10, 3], np.int64)
    v0, c0 = ref.pipeline_partition(tri, xfer, 2, 0)
    v1, c1 = ref.pipeline_partition(tri, xfer, 2, 1)
    assert v0 == G["toy_sum_best"] and v1 == G["toy_max_best"] and c0.tolist() == c1.tolist() == [0, G["toy_cut"], 3]
    # the last stage's right boundary has no transfer: one stage costs C(0,3) alone
    assert ref.pipeline_partition(tri, xfer, 1, 0)[0] == 16


def test_partition_tie_break_smallest_cut_from_the_back():
    """all stage costs equal: every cut set ties; back-tracking from the last stage takes the smallest start each time"""
    L = 7
    tri = np.full((L, L + 1), -1, np.int64)
    for a in range(L):
        tri[a, a + 1:] = 4
    xfer = np.zeros(L, np.int64)
    for stages in (2, 3, 5):
        val, cuts = ref.pipeline_partition(tri, xfer, stages, 1)
        assert val == 4 and cuts.tolist() == list(range(stages)) + [L]


def test_stage_transfer_hand_value():
    mesh = ref.make_mesh((4, 8), (cf.INTER, cf.INTRA))
    layers = np.zeros(3, dtype=cf.LAYER_DTYPE)
    layers[0] = cf.gemm(64, 64, 64, 2, 4, 18)
    layers[1] = cf.gemm(1001, 777, 512, 2, 4, 18)                 # input 1001 x 777, 2 bytes
    layers[2] = cf.gemm(1001, 512, 512, 4, 4, 18, in_rows=1001, in_cols=777)
    x = ref.stage_transfer(layers, mesh, ref.make_net(cf.ALPHA_PS, (3, 40)))
    assert x[0] == 0 and x[1] == G["xfer_m1"]
    assert x[2] == 2 * (20_000_000 + -(-1001 * 777 * 4 // 32) * 40)  # the consumer's element size
    x3 = ref.stage_transfer(layers, mesh, ref.make_net(cf.ALPHA_PS, (3, 40), micro_batches=3))
    assert x3[1] == G["xfer_m3"]


def test_segment_strategies_reevaluate_and_match_the_triangle():
    rng = np.random.default_rng(5)
    for (L, K) in [(6, 6), (9, 36)]:
        T, node, mask = _random_problem(rng, L, K, hi=7)
        tri = ref.segment_optima(T, node, mask)
        for cuts in ([0, L], [0, 2, L], [0, 1, 2, L], [0, L - 1, L]):
            sc, st = ref.segment_strategies(T, node, mask, cuts)
            for k, (a, b) in enumerate(zip(cuts[:-1], cuts[1:])):
                assert sc[k] == tri[a, b]
                assert ref.chain_cost(_segment_as_chain(T, node, mask, a, b), st[a:b]) == sc[k]
        # one stage: exactly the chain DP's strategy (same tie-breaks)
        _, st = ref.segment_strategies(T, node, mask, [0, L])
        assert st.tolist() == ref.chain_dp(_segment_as_chain(T, node, mask, 0, L)[None])[1][0].tolist()


def test_more_stages_on_smaller_sub_meshes_config3():
    """the outer enumeration over stage counts (Table 3 'Opt. Stages'): stage count P runs every stage on a sub-mesh
    with 1/P of the nodes; the sum objective of one stage equals the plain optimum, and all values are finite"""
    w = cf.config3_transformer24()
    vals = {}
    for stages in (1, 2, 4):
        sub = cf.Workload(w.name, w.layers[:, :40], cf.Mesh((w.mesh.size[0] // stages, w.mesh.size[1]), w.mesh.link), w.net, S=1)
        T, node, mask = _tables(sub)
        tri = ref.segment_optima(T, node, mask)
        xfer = ref.stage_transfer(sub.layers[0], ref.mesh_of(sub), ref.net_of(sub))
        vals[stages], cuts = ref.pipeline_partition(tri, xfer, stages, 1)
        assert vals[stages] < PEN
    sub = cf.Workload(w.name, w.layers[:, :40], w.mesh, w.net, S=1)
    assert vals[1] == ref.chain_dp(ref.build_tables(sub.layers, ref.mesh_of(sub), ref.net_of(sub))[0])[0][0]
