"""Pins of the oracle on meshes with four and five levels (R26): machines such as 2 nodes x 8 GPUs (2 | 2.2.2)
or the paper's 2 nodes x 16 GPUs (2 | 2.2.2.2) refined into prime sub-levels, searched over the matmul
rows {0, 1, 2} of PAPER.md:193 per sub-level.  There the signature index is a mixed-radix number over the ALLOWED rows
only (K = 3^4 = 81, 3^5 = 243), level 0 most significant.  No GPU.

  D1  a level of size 1 changes nothing: the tables of (2, 1, 2, 2) / (1, 2, 2, 1, 2) equal, cell by cell, the three-level
      tables of (2, 2, 2) in the base-6 indexing that R1 / R24 pin (whatever row the size-1 level takes)
  D2  the decode: signature j lists the allowed rows in lexicographic order, per-level triples verbatim PAPER.md:193
  D3  data parallelism (row 0 on every level) in closed form from Table 2
  D4  PAPER.md:203 on 2 x 16 GPUs: a tensor split inside a node is gathered over NVLink only, one split across the nodes
      over the network only
  D5  exhaustive search over K^L strategies equals the DP on an 81-signature chain
  D6  K is bounded: more than 256 signatures, or more than five levels, is refused
  D7  the qualitative result the paper reports for VGG13 on 32 GPUs (Fig. 8): the optimum keeps the weight
      matrices of the three dense layers un-replicated (no B state: zero weight-gradient synchronisation) and runs the early
      convolutions purely data parallel, (S0: p) in and out
"""
import itertools

import numpy as np
import pytest

from oracle import ref
from paper_2301_06813_b200 import configs as cf

ROWS012 = 0x07 << 8
S0, S1, B, P = 0, 1, 2, 3
TRIPLE = [(S0, B, S0), (B, S1, S1), (S1, S0, P), (B, B, B), (P, B, P), (B, P, P)]      # (I, W, O) per row, R1


def _chain(L, seed, attn_at=()):
    rng = np.random.default_rng(seed)
    lay = np.zeros((1, L), dtype=cf.LAYER_DTYPE)
    dims = [int(x) for x in rng.integers(96, 3000, L + 1)]
    for l in range(L):
        if l in attn_at:
            lay[0, l] = cf.attn(640, dims[l], dims[l], 2, 8, 16)
            dims[l + 1] = dims[l]
        else:
            lay[0, l] = cf.gemm(640, dims[l], dims[l + 1], 2, 4, 18, max_rows=8 if l % 2 == 0 else None)
    return lay


def _embed(sizes3, links3, pos_of_ones):
    """insert size-1 levels (any link class, rows {0,1,2}) at the given positions of the final mesh"""
    D = len(sizes3) + len(pos_of_ones)
    sizes, links, src = [], [], 0
    for d in range(D):
        if d in pos_of_ones:
            sizes.append(1); links.append((d & 1) | ROWS012)
        else:
            sizes.append(sizes3[src]); links.append(links3[src] | ROWS012); src += 1
    return tuple(sizes), tuple(links)


# ---- D1 ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ones", [(1,), (0,), (3,), (0, 3), (1, 2), (2, 4)])
def test_size_one_levels_change_nothing(ones):
    sizes3, links3 = (2, 4, 2), (1, 0, 0)
    net = ref.make_net(cf.ALPHA_PS, (3, 40), 3 * 10**7, micro_batches=3)
    sizes, links = _embed(sizes3, links3, ones)
    D = len(sizes)
    mesh = ref.make_mesh(sizes, links)
    K = ref.num_signatures(mesh)
    assert K == 3 ** D
    # compact index -> rows per level -> base-6 index over the three real levels
    to3 = np.zeros(K, np.int64)
    plain = []                                                   # signatures whose size-1 levels take row 0 or 1
    for j, rows in enumerate(itertools.product(range(3), repeat=D)):
        real = [rows[d] for d in range(D) if d not in ones]
        to3[j] = real[0] * 36 + real[1] * 6 + real[2]
        if all(rows[d] < 2 for d in ones):
            plain.append(j)
    plain = np.array(plain)
    for attn_at in ((), (1,)):
        lay = _chain(3, 5, attn_at=attn_at)
        T3, n3, m3 = ref.build_tables(lay, ref.make_mesh(sizes3, [l | ROWS012 for l in links3]), net)
        T, n, m = ref.build_tables(lay, mesh, net)
        assert T.shape == (1, 3, K, K)
        want, wn, wm = T3[:, :, to3[:, None], to3[None, :]], n3[:, :, to3], m3[:, :, to3]
        # GEMM chains: every row of the size-1 level; with an attention layer (no row 2, PAPER.md:189 / R1): rows 0, 1
        sel = np.arange(K) if not attn_at else plain
        assert np.array_equal(T[:, :, sel[:, None], sel[None, :]], want[:, :, sel[:, None], sel[None, :]])
        assert np.array_equal(n[:, :, sel], wn[:, :, sel]) and np.array_equal(m[:, :, sel], wm[:, :, sel])
        assert 0 < m.sum() < m.size and (T < (1 << 50)).any() and (T >= (1 << 50)).any()


# ---- D2 ---------------------------------------------------------------------------------------------------
def test_decode_is_lexicographic_over_allowed_rows():
    allow = [0b000111, 0b001011, 0b110000, 0b000101]          # 3, 3, 2, 2 rows: K = 36
    rows = [[g for g in range(6) if a >> g & 1] for a in allow]
    mesh = ref.make_mesh((2, 3, 2, 5), [(d & 1) | (a << 8) for d, a in enumerate(allow)])
    assert ref.num_signatures(mesh) == 36
    for j, combo in enumerate(itertools.product(*rows)):
        v, I, W, O = ref.sig_states(0, j, mesh)
        assert v == 1
        assert [(I[d], W[d], O[d]) for d in range(4)] == [TRIPLE[g] for g in combo], (j, combo)
    # five levels, paper rows: the last level is the least significant digit
    mesh5 = ref.make_mesh((2, 2, 2, 2, 2), [1 | ROWS012] + [ROWS012] * 4)
    assert ref.num_signatures(mesh5) == 243
    assert ref.sig_states(0, 1, mesh5)[1] == (S0, S0, S0, S0, B)
    assert ref.sig_states(0, 2 * 81, mesh5)[3] == (P, S0, S0, S0, S0)
    assert ref.sig_states(1, 2, mesh5)[0] == 0                  # attention has no row 2


# ---- D3 ---------------------------------------------------------------------------------------------------
def test_data_parallel_closed_form_on_five_levels():
    sizes, links = (2, 2, 2, 2, 2), (1, 0, 0, 0, 0)
    alpha, beta = (2_000_000, 9_000_000), (4, 37)
    mesh = ref.make_mesh(sizes, [l | ROWS012 for l in links])
    net = ref.make_net(alpha, beta, 0)
    Kd, N = 1000, 3001
    lay = np.zeros((1, 2), dtype=cf.LAYER_DTYPE)
    lay[0, 0] = cf.gemm(4096, 555, Kd, 2, 4, 18)
    lay[0, 1] = cf.gemm(4096, Kd, N, 2, 4, 18)
    T, node, mask = ref.build_tables(lay, mesh, net)
    nbytes = Kd * N * 4                                          # W replicated everywhere: the whole gradient
    want = 0
    for p, c in zip(sizes, links):
        want += (2 * p - 1) * alpha[c] + 2 * (p - 1) * -(-nbytes // p) * beta[c]
    assert node[0, 1, 0] == want
    assert T[0, 1, 0, 0] == want                                 # S0 -> S0 on every level: no redistribution
    assert mask[0, 1, 0] == 1


# ---- D4 ---------------------------------------------------------------------------------------------------
def test_intra_node_gather_uses_nvlink_only():
    sizes, links = (2, 2, 2, 2, 2), (1, 0, 0, 0, 0)             # 2 nodes | 16 GPUs
    alpha, beta = (2_000_000, 9_000_000), (4, 37)
    mesh = ref.make_mesh(sizes, [l | ROWS012 for l in links])
    net = ref.make_net(alpha, beta, 0)
    rows, cols, eb = 4096, 1024, 2
    n = rows * cols * eb
    allB = (B,) * 5
    for d in range(5):
        a = tuple(S0 if e == d else B for e in range(5))
        c = links[d]
        assert ref.reshard(rows, cols, eb, a, allB, mesh, net) == alpha[c] + (n // 2) * beta[c]      # AllGather, p = 2
    # split over two intra-node levels: gathered outermost first, (p-1)/p of the OUTPUT of each step
    a = (B, B, S0, B, S0)
    assert ref.reshard(rows, cols, eb, a, allB, mesh, net) == (alpha[0] + (n // 4) * beta[0]) + (alpha[0] + (n // 2) * beta[0])


# ---- D5 ---------------------------------------------------------------------------------------------------
def test_exhaustive_search_equals_dp_at_k81():
    mesh = ref.make_mesh((2, 2, 2, 2), [1 | ROWS012, ROWS012, ROWS012, ROWS012])
    net = ref.make_net(cf.ALPHA_PS, (3, 40), 0)
    lay = _chain(2, 11)
    T, _, _ = ref.build_tables(lay, mesh, net)
    assert T.shape[-1] == 81
    cost = T[0, 0, 0][:, None] + T[0, 1]                         # Cost((i, j)) = T[0][0][i] + T[1][i][j]
    best = cost.min()
    i, j = np.argwhere(cost == best)[0]                          # smallest (i, j) in lexicographic order
    dc, ds = ref.chain_dp(T)
    assert dc[0] == best and tuple(ds[0].tolist()) == (i, j)
    bc, bs = ref.brute_force(T[0, :, :9, :9].copy())             # a 9-signature sub-problem through the enumerator
    d9, s9 = ref.chain_dp(T[:, :, :9, :9].copy())
    assert bc == d9[0] and tuple(bs) == tuple(s9[0].tolist())


# ---- D6 ---------------------------------------------------------------------------------------------------
def test_k_is_bounded():
    assert ref.num_signatures(ref.make_mesh((2, 2, 2, 2), (0, 0, 0, 0))) == -1          # 6^4 > 256
    assert ref.num_signatures(ref.make_mesh((2, 2, 2, 2), [0x0f << 8] * 4)) == 256
    assert ref.num_signatures(ref.make_mesh((2, 2, 2, 2, 2), [0x0f << 8] * 5)) == -1
    m = ref.make_mesh((2, 2, 2, 2, 2), [ROWS012] * 5)
    m.ndim = 6
    assert ref.num_signatures(m) == -1


# ---- D7 ---------------------------------------------------------------------------------------------------
def test_vgg13_on_32_nodes_has_the_structure_of_fig8():
    w = cf.CONFIGS[8]()
    mesh, net = ref.mesh_of(w), ref.net_of(w)
    assert ref.num_signatures(mesh) == 243 and w.L == 13
    T, node, mask = ref.build_tables(w.layers, mesh, net)
    dc, ds = ref.chain_dp(T)
    assert dc[0] < (1 << 50)
    strat = ds[0].tolist()
    for l in (10, 11, 12):                                       # dense layers: "W1, W2, and W3 are not replicated"
        _, I, W, O = ref.sig_states(0, strat[l], mesh)
        assert B not in W, (l, W)
        assert node[0, l, strat[l]] == 0                         # "zero weight gradient synchronization overhead"
    for l in range(6):                                           # convolutions: "(S0: p) for input and output tensors"
        assert strat[l] == 0
        _, I, W, O = ref.sig_states(0, 0, mesh)
        assert set(I) == {S0} and set(O) == {S0} and set(W) == {B}
    # data parallelism throughout is not even feasible here (the first dense layer's replicated weight state alone
    # exceeds the per-layer share of 16 GB) and the best 1-opt strategies CD finds are no better than the optimum
    assert ref.chain_cost(T[0], [0] * w.L) >= (1 << 50)
    cc, cs, _ = ref.coord_descent(T, w.cd_init(), w.max_sweeps)
    assert (cc >= dc[0]).all() and cc.min() < (1 << 50)


# ---- stored optima of the extra configs (regression values written by tests/golden/make_extra_config_optima.py) ----------
@pytest.mark.parametrize("k", [6, 7, 8])
def test_stored_optima_of_the_extra_configs(k):
    from tests.conftest import read_golden
    g = read_golden("extra_config_optima.txt")
    w = cf.CONFIGS[k]()
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    dc, ds = ref.chain_dp(T)
    assert int(dc[0]) == g["config%d_dp" % k]
    assert sum((l + 1) * int(s) for l, s in enumerate(ds[0])) == g["config%d_strategy_sum" % k]
