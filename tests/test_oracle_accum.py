"""Pins of gradient accumulation in the cost tables (R25; "divides each mini-batch into micro-batches
and accumulates their gradients", :325 "only communicate the entire model gradients when a mini-batch is complete").
With m micro-batches the redistribution term of every cell is paid m times, the weight-gradient term once.  No GPU."""
import numpy as np

from oracle import ref
from paper_2301_06813_b200 import configs as cf

PEN = 1 << 50


def _tables(w, m):
    net = ref.make_net(w.net.alpha_ps, w.net.beta_ps_per_byte, w.net.mem_cap_bytes, m)
    return ref.build_tables(w.layers, ref.mesh_of(w), net)


def test_cells_are_m_times_edge_plus_node():
    for w in (cf.config1_tiny(), cf.config3_transformer24(), cf.config4_batched(Bp=2, L=5)):
        T1, node1, mask1 = _tables(w, 1)
        T0, _, _ = _tables(w, 0)
        assert np.array_equal(T0, T1)                                    # 0 and 1 both mean no accumulation
        for m in (2, 7, 64):
            Tm, nodem, maskm = _tables(w, m)
            assert np.array_equal(nodem, node1) and np.array_equal(maskm, mask1)     # gradients once per mini-batch
            pen = np.where(mask1[:, :, None, :] == 1, 0, PEN)
            edge1 = T1 - node1[:, :, None, :] - pen                       # the redistribution part of every cell
            assert (edge1 >= 0).all()
            assert np.array_equal(Tm, m * edge1 + node1[:, :, None, :] + pen)
            assert np.array_equal(Tm[:, 0], T1[:, 0])                     # first layer: no producer, nothing to redistribute


def test_hand_cell_and_data_parallel_limit():
    w = cf.config1_tiny()
    T1, _, _ = _tables(w, 1)
    T5, _, _ = _tables(w, 5)
    assert T1[0, 1, 14, 7] == 106_029_312 and T5[0, 1, 14, 7] == 5 * 106_029_312       # tests/golden/hand_cells.txt, node 0
    # pure data parallelism (all signature 0) redistributes nothing: its cost does not depend on m ...
    dp_cost = ref.chain_cost(T1[0], [0] * w.L)
    assert dp_cost == 1_021_420_288
    for m in (1, 5, 1000):
        Tm, _, _ = _tables(w, m)
        assert ref.chain_cost(Tm[0], [0] * w.L) == dp_cost
    # ... so the optimum is non-decreasing in m and can never exceed the data-parallel cost
    prev = 0
    for m in (1, 2, 5, 50, 1000, 10**6):
        Tm, _, _ = _tables(w, m)
        c, s = ref.chain_dp(Tm)
        assert prev <= c[0] <= dp_cost
        prev = int(c[0])
    # ... and for m large enough only redistribution-free strategies survive
    Tm, _, _ = _tables(w, 10**6)
    c, s = ref.chain_dp(Tm)
    T1c = ref.chain_cost(T1[0], s[0])
    assert c[0] == T1c                                                    # same cost under m = 1: every edge on the path is 0
