"""The folded factorisation space on the GPU (R28; up to eight mesh levels, one signature per ordered
factorisation) against the oracle, bit for bit: tables, node costs, masks, chain DP, Coordinate Descent and the one-call
path -- on the paper's Piz Daint Transformer at 64 / 128 / 256 single-GPU nodes and on random meshes."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref
from paper_2301_06813_b200 import configs as cf

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def adl():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_2301_06813_b200 import binding
    binding.lib()
    return binding


def _check(adl, w, init, cap_sw=64):
    dl = adl.layers_to_device(w.layers)
    dinit = torch.from_numpy(init).cuda()
    assert adl.num_signatures(w.mesh) == w.K
    T, node, mask = adl.build_tables(dl, w.mesh, w.net)
    work = torch.empty(adl.workspace_bytes(w.Bp, w.L, w.S, w.mesh), dtype=torch.uint8, device="cuda")
    dc, ds = adl.chain_dp(T, w.mesh, work=work)
    cc, cs, sw = adl.coord_descent(T, dinit, w.mesh, cap_sw)
    o = adl.search(dl, w.mesh, w.net, init=dinit, max_sweeps=cap_sw, want_node_mask=True)
    torch.cuda.synchronize()
    oT, on, om = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    odc, ods = ref.chain_dp(oT)
    occ, ocs, osw = ref.coord_descent(oT, init, cap_sw)
    for name, g, x in (("T", T, oT), ("node", node, on), ("mask", mask, om), ("dp_cost", dc, odc), ("dp_strategy", ds, ods),
                       ("cd_cost", cc, occ), ("cd_strategy", cs, ocs), ("cd_sweeps", sw, osw),
                       ("search.T", o["T"], oT), ("search.node", o["node"], on), ("search.mask", o["mask"], om),
                       ("search.dp_cost", o["opt_cost"], odc), ("search.dp_strategy", o["strategy"], ods),
                       ("search.cd_cost", o["cd_cost"], occ), ("search.cd_strategy", o["cd_strategy"], ocs), ("search.cd_sweeps", o["cd_sweeps"], osw)):
        assert np.array_equal(g.cpu().numpy(), x), (w.name, name)
    return odc


@pytest.mark.parametrize("k", [9, 10, 11])
def test_piz_daint_transformer(adl, k):
    w = cf.CONFIGS[k]()
    init = w.cd_init()[:, :16]
    opt = _check(adl, cf.Workload(w.name, w.layers, w.mesh, w.net, S=16, seed=w.seed), init)
    assert opt[0] < (1 << 50)                                     # a feasible strategy exists under the 16 GB cap
    # data parallelism (signature 0 everywhere) does not fit 16 GB: 8192^2 weights with optimizer state per layer
    _, _, mask = ref.build_tables(w.layers[:, :5], ref.mesh_of(w), ref.net_of(w))
    assert mask[0, 0, 0] == 0


def test_random_folded_meshes(adl):
    rng = np.random.default_rng(21)
    for case in range(60):
        D = int(rng.integers(1, 9))
        sizes = tuple(int(x) for x in rng.choice([2, 2, 2, 3, 4], D))
        links = [int(rng.integers(0, 2)) for _ in range(D)]
        if rng.random() < 0.6:                                     # long runs of equal levels: few groups
            sizes = tuple(sorted(sizes))
            links = sorted(links, reverse=True)
        mesh = cf.Mesh(sizes, (links[0] | cf.FOLD,) + tuple(links[1:]))
        if mesh.K > 256 or int(np.prod(sizes)) > (1 << 20):
            continue
        Bp = int(rng.choice([1, 2, 7, 40]))
        L = int(rng.choice([1, 2, 3, 5, 9, 17]))
        if Bp * L * mesh.K * mesh.K > 2_000_000:
            Bp = max(1, 2_000_000 // (L * mesh.K * mesh.K))
        layers = cf.config4_batched(Bp=Bp, L=L, seed=int(rng.integers(0, 1000))).layers.copy()
        if rng.random() < 0.5:
            for p in range(Bp):
                for l in range(L):
                    if rng.random() < 0.3:
                        layers[p, l] = cf.attn(int(layers[p, l]["M"]), int(layers[p, l]["N"]), int(rng.integers(1, 4000)), 2,
                                               int(rng.integers(1, 40)), int(rng.integers(1, 40)))
        if rng.random() < 0.3:
            layers["max_split_rows"] = rng.integers(1, 40, size=layers.shape)
            layers["max_split_cols"] = rng.integers(1, 40, size=layers.shape)
        if rng.random() < 0.5:
            layers["in_rows"] = rng.integers(1, 5000, size=layers.shape)
            layers["in_cols"] = rng.integers(1, 5000, size=layers.shape)
        cap = int(rng.choice([0, 0, 10**7 * L, 10**9 * L]))
        w = cf.Workload("folded-%d" % case, layers, mesh, cf.Net(cf.ALPHA_PS, (3, 40), cap, micro_batches=int(rng.choice([0, 1, 3]))),
                        S=int(rng.choice([1, 2, 3])), seed=int(rng.integers(0, 1000)))
        _check(adl, w, w.cd_init(), cap_sw=int(rng.choice([1, 2, 64])))


def test_refusals(adl):
    with pytest.raises(adl.AutoddlError):
        adl.num_signatures(cf.Mesh((2,) * 6, (1,) * 6))            # six levels without the fold bit
    with pytest.raises(adl.AutoddlError):
        adl.num_signatures(cf.Mesh((2, 3, 2, 3, 2, 3, 2, 3), (1 | cf.FOLD, 1, 1, 1, 1, 1, 1, 1)))   # eight groups of one level: 3^8 > 256
    with pytest.raises(adl.AutoddlError):
        adl.num_signatures(cf.Mesh((2, 2), (1, 1 | cf.FOLD)))      # the fold bit lives in link[0]
