"""Pins of the restricted signature space (R24): with rows {0, 1, 2} allowed on every level of a mesh refined
into prime sub-levels, the strategies are exactly the paper's SBP matmul factorisations
  I = (S0: p0, B: p1, S1: p2),  W = (B, S1, S0),  O = (S0, S1, P),  p = p0 p1 p2,
with (nodes, GPUs) tuples per SBP dimension.  No GPU."""
import itertools

import numpy as np

from oracle import ref
from paper_2301_06813_b200 import configs as cf

PAPER_ROWS = 0x07 << 8          # rows 0, 1, 2


def _mesh(sizes, links, allow=PAPER_ROWS):
    return ref.make_mesh(sizes, [l | allow for l in links])


def _layers(L, M=512, H=768):
    out = np.zeros((1, L), dtype=cf.LAYER_DTYPE)
    for l in range(L):
        out[0, l] = cf.gemm(M, H, H, 2, 4, 18)
    return out


def test_feasible_set_is_the_factorisation_space():
    """8 nodes x 1 GPU = 2.2.2 (PAPER.md:201 Multi-Node-Single-GPU): 27 assignments = the 10 ordered factorisations
    p0 p1 p2 = 8 counted with the multiplicity of placing the prime factors"""
    mesh = _mesh((2, 2, 2), (1, 1, 1))
    net = ref.make_net(cf.ALPHA_PS, (3, 40), 0)
    lay = _layers(1)
    T, node, mask = ref.build_tables(lay, mesh, net)
    ok = np.flatnonzero(mask[0, 0])
    want = [a * 36 + b * 6 + c for a, b, c in itertools.product(range(3), repeat=3)]
    assert ok.tolist() == want
    facts = {}
    for j in ok:
        digs = [(j // 36) % 6, (j // 6) % 6, j % 6]
        p = [1, 1, 1]
        for g in digs:
            p[g] *= 2
        facts[tuple(p)] = facts.get(tuple(p), 0) + 1
        v, I, W, O = ref.sig_states(0, int(j), mesh)
        assert v == 1
        for d, g in enumerate(digs):                          # verbatim PAPER.md:193
            assert (I[d], W[d], O[d]) == [(0, 2, 0), (2, 1, 1), (1, 0, 3)][g]    # S0 = 0, S1 = 1, B = 2, P = 3
    assert len(facts) == 10 and sum(facts.values()) == 27 and facts[(2, 2, 2)] == 6 and facts[(8, 1, 1)] == 1
    # every other column carries the penalty, every allowed one the unrestricted value
    Tu, _, masku = ref.build_tables(lay, ref.make_mesh((2, 2, 2), (1, 1, 1)), net)
    assert np.array_equal(T[..., ok], Tu[..., ok])
    bad = np.setdiff1d(np.flatnonzero(masku[0, 0]), ok)
    assert len(bad) > 0 and np.array_equal(T[..., bad], Tu[..., bad] + (1 << 50))


def test_link_class_is_bit_zero_only():
    """the allow bits do not leak into the link class: costs of allowed cells equal the unrestricted ones"""
    net = ref.make_net(cf.ALPHA_PS, (3, 40), 0)
    lay = _layers(3)
    for sizes, links in (((4, 2), (1, 0)), ((2, 2, 2), (1, 0, 0)), ((8,), (1,))):
        Tr, _, mr = ref.build_tables(lay, _mesh(sizes, links), net)
        Tu, _, mu = ref.build_tables(lay, ref.make_mesh(sizes, links), net)
        ok = mr.astype(bool)
        assert ok.sum() == 3 * 3 ** len(sizes)
        sel = np.broadcast_to(ok[:, :, None, :], Tr.shape)
        assert np.array_equal(Tr[sel], Tu[sel])


def test_optimum_over_the_paper_space():
    """exhaustive search over the 27^L factorisation strategies (the paper's own optimum) equals the DP on the
    restricted tables; the restricted optimum is feasible, uses allowed signatures only and is >= the unrestricted one"""
    net = ref.make_net(cf.ALPHA_PS, (3, 40), 0)
    rng = np.random.default_rng(3)
    L = 3
    lay = np.zeros((1, L), dtype=cf.LAYER_DTYPE)
    dims = [int(x) for x in rng.integers(64, 4096, L + 1)]
    for l in range(L):
        lay[0, l] = cf.gemm(777, dims[l], dims[l + 1], 2, 4, 18)
    mesh = _mesh((2, 2, 2), (1, 1, 0))
    T, _, mask = ref.build_tables(lay, mesh, net)
    allowed = [a * 36 + b * 6 + c for a, b, c in itertools.product(range(3), repeat=3)]
    best = None
    for s in itertools.product(allowed, repeat=L):
        c = ref.chain_cost(T[0], s)
        if best is None or c < best[0]:
            best = (c, s)
    dc, ds = ref.chain_dp(T)
    assert dc[0] == best[0] and tuple(ds[0].tolist()) == best[1] and dc[0] < (1 << 50)
    Tu, _, _ = ref.build_tables(lay, ref.make_mesh((2, 2, 2), (1, 1, 0)), net)
    du, _ = ref.chain_dp(Tu)
    assert du[0] <= dc[0]
    # data parallelism (all p1 = p2 = 1) is in the space and costs what it cost before
    assert ref.chain_cost(T[0], [0] * L) == ref.chain_cost(Tu[0], [0] * L)
    # coordinate descent started inside the space stays inside it
    init = np.array([[[allowed[5], allowed[20], allowed[11]], [0, 0, 0]]], np.int32)
    cc, cs, _ = ref.coord_descent(T, init)
    assert (cc < (1 << 50)).all() and np.isin(cs, allowed).all() and (cc >= dc[0]).all()
