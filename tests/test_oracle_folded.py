"""Pins of the oracle's FOLDED factorisation space (R28; PAPER.md:193 p = p0 p1 p2, :201 (nodes, GPUs) tuples), no
GPU.  A signature is an ordered factorisation per group of equal mesh levels = the canonical (sorted) digit string of
the prime-sub-level encoding (R24 / R26); so on every machine BOTH encodings express the folded tables must equal the
canonical rows / columns of the prime tables cell by cell; beyond five levels only the folded space exists and is
pinned by the decode order (enumeration), closed forms and hand cells (tests/golden/folded_hand_values.txt)."""
import itertools

import numpy as np
import pytest

from oracle import ref
from paper_2301_06813_b200 import configs as cf
from tests.conftest import read_golden

S0, S1, B, P = 0, 1, 2, 3
ROWS = {0: (S0, B, S0), 1: (B, S1, S1), 2: (S1, S0, P)}          # (I, W, O) of the paper's three factors
G = read_golden("folded_hand_values.txt")
A = cf.PAPER_ROWS


def _groups(mesh):
    out, d = [], 0
    while d < mesh.ndim:
        n = 1
        while d + n < mesh.ndim and mesh.size[d + n] == mesh.size[d] and (mesh.link[d + n] & 1) == (mesh.link[d] & 1):
            n += 1
        out.append(n)
        d += n
    return out


def _canonical_strings(mesh):
    """all signatures of the folded space as digit strings, in index order: per group the sorted strings in increasing
    lexicographic order, group 0 most significant -- by enumeration of all 3^n strings"""
    per_group = [[s for s in itertools.product(range(3), repeat=n) if list(s) == sorted(s)] for n in _groups(mesh)]
    return [sum(parts, ()) for parts in itertools.product(*per_group)]


def _fold(mesh):
    return cf.Mesh(mesh.size, ((mesh.link[0] & 1) | cf.FOLD,) + tuple(l & 1 for l in mesh.link[1:]))


MESHES = [cf.Mesh((2, 2, 2), (1 | A, 1 | A, 1 | A)), cf.Mesh((2, 2, 2, 2), (1 | A,) * 4), cf.Mesh((2,) * 5, (1 | A,) * 5),
          cf.Mesh((2, 2, 2, 2), (1 | A, A, A, A)), cf.Mesh((2, 2, 2, 2, 2), (1 | A, 1 | A, A, A, A)), cf.Mesh((3, 3, 2, 2), (1 | A, 1 | A, A, A)),
          cf.Mesh((2, 2), (1 | A, 1 | A)), cf.Mesh((4, 2, 2), (1 | A, A, A))]


@pytest.mark.parametrize("n", [1, 2, 3, 6, 7, 8])
def test_decode_order_and_count(n):
    mesh = cf.Mesh((2,) * n, (cf.INTER | cf.FOLD,) + (cf.INTER,) * (n - 1))
    rm = ref.mesh_of(cf.Workload("x", np.zeros((1, 1), cf.LAYER_DTYPE), mesh, cf.Net(), 1))
    strings = _canonical_strings(mesh)
    assert ref.num_signatures(rm) == len(strings) == (n + 2) * (n + 1) // 2 == mesh.K
    for j, s in enumerate(strings):
        v, I, W, O = ref.sig_states(cf.GEMM, j, rm)
        assert v == 1 and (I, W, O) == tuple(zip(*[ROWS[g] for g in s])), (j, s)
    # the factorisation it stands for: p0 = 2^#0, p1 = 2^#1, p2 = 2^#2, in decreasing p0 then decreasing p1
    facts = [(2 ** s.count(0), 2 ** s.count(1), 2 ** s.count(2)) for s in strings]
    assert facts == sorted(facts, reverse=True) and all(a * b * c == 2 ** n for a, b, c in facts)


def test_counts_of_the_papers_machines():
    assert cf.Mesh((2,) * 6, (1 | cf.FOLD,) + (1,) * 5).K == 28 and cf.Mesh((2,) * 8, (1 | cf.FOLD,) + (1,) * 7).K == 45
    two_by_16 = cf.Mesh((2, 2, 2, 2, 2), (1 | cf.FOLD, 0, 0, 0, 0))     # (nodes, GPUs) tuples
    assert two_by_16.K == 3 * 15 and ref.num_signatures(ref.make_mesh(two_by_16.size, two_by_16.link)) == 45
    assert ref.num_signatures(ref.make_mesh((2,) * 6, (1,) * 6)) == -1  # six levels exist only in the folded space


@pytest.mark.parametrize("mesh", MESHES, ids=lambda m: "x".join(map(str, m.size)) + "_" + "".join(str(l & 1) for l in m.link))
def test_folded_tables_equal_canonical_prime_tables(mesh):
    """every machine both encodings express: the folded table is the sub-table of the prime-sub-level table on the
    canonical signatures -- T, node and mask, cell by cell, ragged dims, an attention layer and a memory cap included"""
    rng = np.random.default_rng(sum(mesh.size))
    L = 5
    layers = np.zeros((2, L), dtype=cf.LAYER_DTYPE)
    for p in range(2):
        for l in range(L):
            M, Kd, N = (int(x) for x in rng.integers(1, 3000, 3))
            layers[p, l] = (cf.attn(M, N, int(rng.integers(1, 3000)), 2, int(rng.integers(1, 40)), int(rng.integers(1, 40))) if l == 2 else
                            cf.gemm(M, Kd, N, 2, 4, 18, in_rows=int(rng.integers(1, 5000)), in_cols=int(rng.integers(1, 5000)),
                                    max_rows=int(rng.integers(1, 64)), max_cols=int(rng.integers(1, 64))))
    net = cf.Net(cf.ALPHA_PS, (3, 40), 400_000 * L, micro_batches=3)
    wp = cf.Workload("prime", layers, mesh, net, S=1)
    wf = cf.Workload("folded", layers, _fold(mesh), net, S=1)
    Tp, np_, mp_ = ref.build_tables(wp.layers, ref.mesh_of(wp), ref.net_of(wp))
    Tf, nf, mf = ref.build_tables(wf.layers, ref.mesh_of(wf), ref.net_of(wf))
    strings = _canonical_strings(mesh)
    radix = 6 if mesh.ndim <= 3 else 3                            # R1 base-6 index up to three levels, R26 over rows {0,1,2} beyond
    canon = [sum(g * radix ** (mesh.ndim - 1 - d) for d, g in enumerate(s)) for s in strings]
    assert Tf.shape[-1] == len(canon) == wf.K
    assert np.array_equal(Tf, Tp[:, :, canon][:, :, :, canon])
    assert np.array_equal(nf, np_[:, :, canon]) and np.array_equal(mf, mp_[:, :, canon])
    # the search over the folded space is a search over a subset of the prime space: its optimum cannot be better
    assert (ref.chain_dp(Tf)[0] >= ref.chain_dp(Tp)[0]).all()


@pytest.mark.parametrize("n", [6, 7, 8])
def test_data_parallel_closed_form_beyond_five_levels(n):
    mesh = cf.Mesh((2,) * n, (cf.INTER | cf.FOLD,) + (cf.INTER,) * (n - 1))
    lay = np.zeros((1, 2), dtype=cf.LAYER_DTYPE)
    lay[0, 0] = cf.gemm(4096, 8192, 8192, 4, 4, 16)
    lay[0, 1] = cf.gemm(4096, 8192, 8192, 4, 4, 16)
    w = cf.Workload("dp", lay, mesh, cf.Net(cf.ALPHA_PS, (3, 40), 0), S=1)
    T, node, mask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    assert node[0, 0, 0] == G["dp_node_%d_levels" % n]
    assert T[0, 1, 0, 0] == G["dp_node_%d_levels" % n]            # data parallel -> data parallel: no redistribution
    assert node[0, 0, w.K - 1] == 0                               # (1, 1, p): W split on the reduction dim everywhere
    assert mask.all()


def test_hand_cell_gather_over_six_levels():
    mesh = cf.Mesh((2,) * 6, (cf.INTER | cf.FOLD,) + (cf.INTER,) * 5)
    rm = ref.make_mesh(mesh.size, mesh.link)
    net = ref.make_net(cf.ALPHA_PS, (3, 40))
    strings = _canonical_strings(mesh)
    j_allB = strings.index((1,) * 6)                              # (1, 64, 1): I = B on every level
    assert ref.sig_states(cf.GEMM, j_allB, rm)[1] == (B,) * 6 and ref.sig_states(cf.GEMM, 0, rm)[3] == (S0,) * 6
    prev = cf.gemm(4096, 512, 1024, 2, 4, 18)
    cur = cf.gemm(4096, 1024, 512, 2, 4, 18)
    assert ref.edge_cost(prev, cur, 0, j_allB, rm, net) == G["edge_dp_to_allB"]


def test_exhaustive_search_equals_dp_on_the_folded_space():
    mesh = cf.Mesh((2, 2, 2), (cf.INTER | cf.FOLD, cf.INTER, cf.INTER))     # 8 nodes: 10 ordered factorisations
    w = cf.config4_batched(Bp=3, L=4, seed=8)
    w = cf.Workload("f", w.layers, mesh, w.net, S=1)
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    assert T.shape[-1] == 10
    dc, ds = ref.chain_dp(T)
    for p in range(3):
        bc, bs = ref.brute_force(T[p])                            # 10^4 strategies
        assert bc == dc[p] and ref.chain_cost(T[p], ds[p]) == dc[p]
