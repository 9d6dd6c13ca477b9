"""Parity on meshes with four and five levels (R26: the signature index runs over the allowed rows only,
K <= 256; 2 nodes x 8 GPUs = 2 | 2.2.2, the paper's 2 nodes x 16 GPUs = 2 | 2.2.2.2): every path of the
CUDA library against the oracle, bit-exact.  `pytest -m gpu`."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref
from paper_2301_06813_b200 import configs as cf

pytestmark = pytest.mark.gpu
PAPER = 0x07 << 8


@pytest.fixture(scope="module")
def adl():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_2301_06813_b200 import binding
    binding.lib()
    return binding


def _workload(Bp, L, sizes, links, seed, S=2, attn=False, cap=0, micro=1):
    w = cf.config4_batched(Bp=Bp, L=L, seed=seed)
    layers = w.layers.copy()
    if attn:
        for p in range(Bp):
            for l in range(1, L, 3):
                layers[p, l] = cf.attn(int(layers[p, l]["M"]), int(layers[p, l]["N"]), int(layers[p, l]["in_cols"]), 2, 8, 16)
    return cf.Workload("deep-mesh", layers, cf.Mesh(sizes, links), cf.Net(cf.ALPHA_PS, (3, 40), cap, micro), S=S, seed=seed)


def _same(got, want, names):
    for g, x, n in zip(got, want, names):
        g = g.cpu().numpy() if hasattr(g, "cpu") else g
        assert g.shape == x.shape and np.array_equal(g, x), n


NAMES = ("T", "node", "mask", "dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps")


@pytest.mark.parametrize("sizes,links,Bp,L,cap,micro", [
    ((2, 2, 2, 2), (1 | PAPER, 0 | PAPER, 0 | PAPER, 0 | PAPER), 3, 6, 0, 1),                      # 2 x 8 GPUs, K = 81
    ((2, 2, 2, 2, 2), (1 | PAPER, 0 | PAPER, 0 | PAPER, 0 | PAPER, 0 | PAPER), 2, 5, 0, 1),       # 2 x 16 GPUs, K = 243
    ((2, 2, 2, 2), (1 | PAPER, 1 | PAPER, 0 | PAPER, 0 | PAPER), 21, 4, 0, 1),                     # 21 chains: one CTA per chain
    ((2, 2, 2, 2), (1 | (0x0f << 8), 0 | PAPER, 0 | PAPER, 0 | (0x03 << 8)), 2, 9, 0, 1),         # K = 72: last cluster CTA owns no row
    ((2, 2, 2, 2, 2), (1 | PAPER, 1 | PAPER, 0 | PAPER, 0 | PAPER, 0 | PAPER), 1, 7, 10**8, 4),   # 4 x 8, cap, accumulation
    ((3, 2, 2, 5), (1 | PAPER, 1 | (0x0b << 8), 0 | (0x30 << 8), 0 | (0x05 << 8)), 2, 6, 0, 1),    # unequal row sets: K = 36
    ((2, 3, 2, 2), (1 | (0x0f << 8), 0 | (0x0f << 8), 0 | (0x0f << 8), 1 | (0x0f << 8)), 1, 3, 0, 2),   # K = 256
    ((2, 1, 4, 2, 1), (1 | (0x03 << 8), 0 | (0x01 << 8), 0 | PAPER, 0 | PAPER, 1 | (0x09 << 8)), 5, 4, 0, 1),   # K = 36
])
def test_every_path(adl, sizes, links, Bp, L, cap, micro):
    w = _workload(Bp, L, sizes, links, seed=len(sizes) + L, attn=True, cap=cap, micro=micro)
    K = w.K
    assert adl.num_signatures(w.mesh) == K == ref.num_signatures(ref.mesh_of(w))
    init = w.cd_init()
    oT, onode, omask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    assert oT.shape[-1] == K and 0 < omask.sum() < omask.size
    odc, ods = ref.chain_dp(oT)
    occ, ocs, osw = ref.coord_descent(oT, init, w.max_sweeps)
    d_layers = adl.layers_to_device(w.layers)
    T, node, mask = adl.build_tables(d_layers, w.mesh, w.net)
    work = torch.empty(adl.workspace_bytes(w.Bp, w.L, w.S, w.mesh), dtype=torch.uint8, device="cuda")
    dc, ds = adl.chain_dp(T, w.mesh, work=work)
    cc, cs, sw = adl.coord_descent(T, torch.from_numpy(init).cuda(), w.mesh, w.max_sweeps)
    _same((T, node, mask, dc, ds, cc, cs, sw), (oT, onode, omask, odc, ods, occ, ocs, osw), NAMES)
    one = adl.search(d_layers, w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=w.max_sweeps, want_node_mask=True)
    _same([one[k] for k in ("T", "node", "mask", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")],
          (oT, onode, omask, odc, ods, occ, ocs, osw), NAMES)
    want = ref.metropolis(oT, init, 1200, 30_000_000, seed=2)
    got = adl.metropolis(T, torch.from_numpy(init).cuda(), w.mesh, 1200, 30_000_000, seed=2)
    _same(got, want, ("best_cost", "best_strategy", "final_cost", "final_strategy", "accepted"))


def test_long_chain_back_pointers_in_the_workspace(adl):
    """L * K > 16 Ki: the any-K DP keeps its back-pointers in the caller's workspace; tables built by the library (d_T NULL)"""
    w = _workload(2, 90, (2, 2, 2, 2, 2), (1 | PAPER,) + (PAPER,) * 4, seed=3, S=3)
    oT, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    odc, ods = ref.chain_dp(oT)
    d_layers = adl.layers_to_device(w.layers)
    work = torch.empty(adl.workspace_bytes(w.Bp, w.L, w.S, w.mesh), dtype=torch.uint8, device="cuda")
    dc, ds = adl.chain_dp(None, w.mesh, net=w.net, d_layers=d_layers, work=work)
    _same((dc, ds), (odc, ods), ("dp_cost", "dp_strategy"))
    init = w.cd_init()
    occ, ocs, osw = ref.coord_descent(oT, init, w.max_sweeps)
    cc, cs, sw = adl.coord_descent(None, torch.from_numpy(init).cuda(), w.mesh, w.max_sweeps, net=w.net, d_layers=d_layers, work=work)
    _same((cc, cs, sw), (occ, ocs, osw), ("cd_cost", "cd_strategy", "cd_sweeps"))


def test_config7_full_size(adl):
    """the paper's 2 x 16 GPU machine on its large Transformer (configs.config7): the whole 140 x 243 x 243 table, the
    optimum, CD from 64 starts and the host-buffer entry point, all against the oracle"""
    w = cf.CONFIGS[7]()
    assert (w.K, w.L) == (243, 140)
    init = w.cd_init()
    oT, onode, omask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    odc, ods = ref.chain_dp(oT)
    occ, ocs, osw = ref.coord_descent(oT, init, w.max_sweeps)
    assert odc[0] < (1 << 50) and ref.chain_cost(oT[0], [0] * w.L) >= (1 << 50)      # data parallelism does not fit
    d_layers = adl.layers_to_device(w.layers)
    one = adl.search(d_layers, w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=w.max_sweeps, want_node_mask=True)
    _same([one[k] for k in ("T", "node", "mask", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")],
          (oT, onode, omask, odc, ods, occ, ocs, osw), NAMES)
    wk = cf.Workload(w.name, w.layers, w.mesh, w.net, S=w.S, seed=w.seed, max_sweeps=w.max_sweeps)
    work = torch.empty(adl.workspace_bytes(w.Bp, w.L, w.S, w.mesh), dtype=torch.uint8, device="cuda")
    host = adl.search_host(wk, init, work)
    _same([host[k] for k in ("opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")], (odc, ods, occ, ocs, osw), NAMES[3:])


def test_config8_vgg13_on_32_nodes(adl):
    """the setting of the paper's Fig. 8 (configs.config8): every output against the oracle; the optimum the GPU returns
    keeps the dense layers' weights un-replicated"""
    w = cf.CONFIGS[8]()
    init = w.cd_init()
    oT, onode, omask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    odc, ods = ref.chain_dp(oT)
    occ, ocs, osw = ref.coord_descent(oT, init, w.max_sweeps)
    one = adl.search(adl.layers_to_device(w.layers), w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=w.max_sweeps,
                     want_node_mask=True)
    _same([one[k] for k in ("T", "node", "mask", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")],
          (oT, onode, omask, odc, ods, occ, ocs, osw), NAMES)
    strat = one["strategy"][0].tolist()
    for l in (10, 11, 12):
        assert int(one["node"][0, l, strat[l]]) == 0            # no weight-gradient all-reduce on the dense layers


def test_limits(adl):
    with pytest.raises(adl.AutoddlError, match="256"):
        adl.num_signatures(cf.Mesh((2, 2, 2, 2), (0, 0, 0, 0)))                       # 6^4 signatures
    with pytest.raises(adl.AutoddlError, match="256"):
        adl.num_signatures(cf.Mesh((2, 2, 2, 2, 2), (0x0f << 8,) * 5))               # 4^5
    with pytest.raises(adl.AutoddlError, match="ndim"):
        adl.num_signatures(cf.Mesh((2,) * 6, (PAPER,) * 6))
    assert adl.num_signatures(cf.Mesh((2, 2, 2, 2), (0x0f << 8,) * 4)) == 256


@pytest.mark.parametrize("K,L,Bp,sizes,links", [
    (81, 400, 2, (2, 2, 2, 2), (PAPER,) * 4),                          # gathered back-pointers outgrow the stage memory
    (243, 800, 1, (2, 2, 2, 2, 2), (PAPER,) * 5),                      # too long for the cluster kernel: one CTA, workspace
    (100, 150, 3, (2, 2, 2, 2), (0x1f << 8, 0x1f << 8, 0x03 << 8, 0x03 << 8)),    # run-time K on the cluster kernel
    (243, 33, 19, (2, 2, 2, 2, 2), (PAPER,) * 5),                      # 19 chains: one CTA per chain
])
def test_single_chain_dp_on_caller_tables(adl, K, L, Bp, sizes, links):
    """(a2) alone on random tables with many exact ties (values in [0, 50)): every DP kernel for K <= 256 takes the same
    smallest-index decisions as the definition"""
    mesh = cf.Mesh(sizes, links)
    assert adl.num_signatures(mesh) == K
    rng = np.random.default_rng(K + L)
    T = rng.integers(0, 50, size=(Bp, L, K, K)).astype(np.int64)
    T[:, :, :, ::7] += 1 << 50                                          # infeasible columns
    odc, ods = ref.chain_dp(T)
    work = torch.empty(adl.workspace_bytes(Bp, L, 1, mesh), dtype=torch.uint8, device="cuda")
    dc, ds = adl.chain_dp(torch.from_numpy(T).cuda(), mesh, work=work)
    _same((dc, ds), (odc, ods), ("dp_cost", "dp_strategy"))
