"""Parity on meshes whose levels restrict the signature rows (R24; rows {0,1,2} = the paper's own SBP matmul
factorisation space): every path of the CUDA library against the oracle, bit-exact.  `pytest -m gpu`."""
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


def _workload(Bp, L, sizes, links, seed, S=2, attn=False, cap=0):
    w = cf.config4_batched(Bp=Bp, L=L, seed=seed)
    layers = w.layers.copy()
    if attn:
        for p in range(Bp):
            for l in range(1, L, 3):
                layers[p, l] = cf.attn(int(layers[p, l]["M"]), int(layers[p, l]["N"]), int(layers[p, l]["in_cols"]), 2, 8, 16)
    return cf.Workload("paper-space", layers, cf.Mesh(sizes, links), cf.Net(cf.ALPHA_PS, (3, 40), cap), S=S, seed=seed)


def _same(got, want, names):
    for g, x, n in zip(got, want, names):
        g = g.cpu().numpy() if hasattr(g, "cpu") else g
        assert g.shape == x.shape and np.array_equal(g, x), n


@pytest.mark.parametrize("sizes,links", [((2, 2, 2), (1 | PAPER, 1 | PAPER, 0 | PAPER)),      # 4 nodes x 2 GPUs, K = 216
                                          ((4, 4), (1 | PAPER, 0 | PAPER)),                   # K = 36, both levels restricted
                                          ((4, 4), (1 | PAPER, 0)),                           # only the node level restricted
                                          ((8,), (1 | (0x0b << 8),)),                         # rows {0, 1, 3} on one level
                                          ((3, 5), (1 | (0x3e << 8), 0 | PAPER))])            # data parallelism forbidden on level 0
def test_three_kernels(adl, sizes, links):
    w = _workload(3, 6, sizes, links, seed=len(sizes), attn=True, cap=40 * 10**9)
    init = w.cd_init()
    oT, onode, omask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    assert 0 < omask.sum() < omask.size
    odc, ods = ref.chain_dp(oT)
    occ, ocs, osw = ref.coord_descent(oT, init, w.max_sweeps)
    d_layers = adl.layers_to_device(w.layers)
    T, node, mask = adl.build_tables(d_layers, w.mesh, w.net)
    work = torch.empty(adl.workspace_bytes(w.Bp, w.L, w.S, w.mesh), dtype=torch.uint8, device="cuda")
    dc, ds = adl.chain_dp(T, w.mesh, work=work)
    cc, cs, sw = adl.coord_descent(T, torch.from_numpy(init).cuda(), w.mesh, w.max_sweeps)
    _same((T, node, mask, dc, ds, cc, cs, sw), (oT, onode, omask, odc, ods, occ, ocs, osw),
          ("T", "node", "mask", "dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
    one = adl.search(d_layers, w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=w.max_sweeps, want_node_mask=True)
    _same([one[k] for k in ("T", "node", "mask", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")],
          (oT, onode, omask, odc, ods, occ, ocs, osw), ("T", "node", "mask", "dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
    want = ref.metropolis(oT, init, 1500, 30_000_000, seed=2)
    got = adl.metropolis(T, torch.from_numpy(init).cuda(), w.mesh, 1500, 30_000_000, seed=2)
    _same(got, want, ("best_cost", "best_strategy", "final_cost", "final_strategy", "accepted"))


def test_fused_kernel_on_the_paper_space(adl):
    """400 chains on a 4 x 4 mesh restricted to the matmul rows: the fused kernel (tables + DP + first CD sweep) and the
    CD kernel on class-representative rows; optimum costs >= the unrestricted ones and never infeasible"""
    w = _workload(400, 9, (4, 4), (1 | PAPER, 0 | PAPER), seed=7, S=2)
    init = (w.cd_init() % 3) * 7                      # starts inside the space: digits in {0,1,2} -> sigs {0, 7, 14}
    d_layers = adl.layers_to_device(w.layers)
    one = adl.search(d_layers, w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=w.max_sweeps, want_node_mask=True)
    idx = np.arange(0, 400, 13)
    ws = cf.Workload(w.name, np.ascontiguousarray(w.layers[idx]), w.mesh, w.net, S=w.S, seed=w.seed)
    oT, onode, omask = ref.build_tables(ws.layers, ref.mesh_of(ws), ref.net_of(ws))
    odc, ods = ref.chain_dp(oT)
    occ, ocs, osw = ref.coord_descent(oT, np.ascontiguousarray(init[idx]), w.max_sweeps)
    _same([one[k][idx] for k in ("T", "node", "mask", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")],
          (oT, onode, omask, odc, ods, occ, ocs, osw), ("T", "node", "mask", "dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
    wu = cf.Workload(w.name, w.layers, cf.Mesh((4, 4), (1, 0)), w.net, S=w.S, seed=w.seed)
    du, _ = adl.chain_dp(adl.build_tables(d_layers, wu.mesh, wu.net)[0], wu.mesh)
    assert (one["opt_cost"] >= du).all() and (one["opt_cost"] < (1 << 50)).all() and (one["cd_cost"] < (1 << 50)).all()
    digits_ok = ((one["strategy"] // 6) < 3) & ((one["strategy"] % 6) < 3)
    assert bool(digits_ok.all())


def test_bad_link_bits_rejected(adl):
    with pytest.raises(adl.AutoddlError, match="link"):
        adl.num_signatures(cf.Mesh((2, 2), (1 | (1 << 15), 0)))
    with pytest.raises(adl.AutoddlError, match="link"):
        adl.num_signatures(cf.Mesh((2, 2), (2, 0)))
