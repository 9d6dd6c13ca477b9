"""The structure the fused kernel builds on, checked on the ORACLE (no GPU): on a two-level mesh the forward + backward
redistribution cost of an edge (Table 2 :102-108; R4, R5) depends on a level's pair of states
(producer output a_d, consumer input b_d) only through one of ten classes, so a 36 x 36 tile holds at most 100 distinct
edge values.  The partition is written out here by hand from R4's phases, not computed from any walk
table:
  nothing to do on the level, tensor split on rows:  (S0,S0) (S0,P) (B,S0)      [B -> S0 keeps its own slice; -> P is a zero fill]
  nothing to do, split on columns:                   (S1,S1) (S1,P) (B,S1)
  nothing to do, not split:                          (B,B) (B,P) (P,P)
  and seven pairs on their own:                      (S0,S1) (S0,B) (S1,S0) (S1,B) (P,S0) (P,S1) (P,B)
A pair of the first three classes costs nothing in either direction but leaves the tensor split differently, which changes
the message sizes of the OTHER level: the classes must not be merged (second test)."""
import itertools

import numpy as np

from oracle import ref
from paper_2301_06813_b200 import configs as cf

S0, S1, B, P = 0, 1, 2, 3
CLASSES = [
    {(S0, S0), (S0, P), (B, S0)}, {(S1, S1), (S1, P), (B, S1)}, {(B, B), (B, P), (P, P)},
    {(S0, S1)}, {(S0, B)}, {(S1, S0)}, {(S1, B)}, {(P, S0)}, {(P, S1)}, {(P, B)},
]
CLS = {pair: k for k, members in enumerate(CLASSES) for pair in members}
DUAL = {S0: S0, S1: S1, B: P, P: B}


def _esym(rows, cols, eb, a, b, mesh, net):
    """forward leg a -> b plus backward leg dual(b) -> dual(a) (R5)"""
    return (ref.reshard(rows, cols, eb, a, b, mesh, net) +
            ref.reshard(rows, cols, eb, tuple(DUAL[x] for x in b), tuple(DUAL[x] for x in a), mesh, net))


MESHES = [((4, 4), (cf.INTER, cf.INTRA)), ((3, 5), (cf.INTER, cf.INTRA)), ((8, 2), (cf.INTRA, cf.INTER)), ((1, 7), (cf.INTER, cf.INTRA))]


def test_sixteen_pairs_are_ten_classes():
    assert len(CLS) == 16 and len(CLASSES) == 10


def test_edge_value_is_a_function_of_the_two_level_classes():
    net = ref.make_net(cf.ALPHA_PS, (3, 40))
    states = list(itertools.product(range(4), repeat=2))
    for (size, link), (rows, cols, eb) in itertools.product(MESHES, [(1001, 777, 2), (4096, 12288, 4), (5, 3, 1)]):
        mesh = ref.make_mesh(size, link)
        seen = {}
        for a in states:
            for b in states:
                key = (CLS[(a[0], b[0])], CLS[(a[1], b[1])])
                v = _esym(rows, cols, eb, a, b, mesh, net)
                assert seen.setdefault(key, v) == v, (size, rows, cols, a, b)
        assert len(seen) == 100


def test_the_ten_classes_cannot_be_merged():
    """every two classes are told apart by some edge on a ragged tensor: 100 is not an over-count"""
    net = ref.make_net(cf.ALPHA_PS, (3, 40))
    mesh = ref.make_mesh((3, 5), (cf.INTER, cf.INTRA))
    reps = [sorted(m)[0] for m in CLASSES]
    table = np.array([[[_esym(1001, 777, 2, (p0[0], p1[0]), (p0[1], p1[1]), mesh, net) for p1 in reps] for p0 in reps],
                      [[_esym(1001, 777, 2, (p1[0], p0[0]), (p1[1], p0[1]), mesh, net) for p1 in reps] for p0 in reps]])
    for u, v in itertools.combinations(range(10), 2):        # as the class of level 0 (table[0]) or of level 1 (table[1])
        assert (table[0][u] != table[0][v]).any() and (table[1][u] != table[1][v]).any(), (u, v)


def test_tile_of_the_library_tables_has_at_most_100_edge_values():
    """the same on whole tiles of the oracle's tables: T[l][i][j] - T[l][0-edge row][j] over a GEMM -> GEMM edge"""
    w = cf.config4_batched(Bp=3, L=4, seed=11)
    T, node, mask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    for p in range(w.Bp):
        for l in range(1, w.L):
            vp = node[p, l] + (1 - mask[p, l].astype(np.int64)) * (1 << 50)
            edge = T[p, l] - vp[None, :]
            assert (edge >= 0).all() and len(np.unique(edge)) <= 100
