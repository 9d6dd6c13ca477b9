"""Parity with gradient accumulation (net.micro_batches, R25): all three table builders (K = 6, 36, 216), the
fused one-call path and the searches on top, against the oracle, bit-exact.  `pytest -m gpu`."""
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


def _with_m(w, m):
    net = cf.Net(w.net.alpha_ps, w.net.beta_ps_per_byte, w.net.mem_cap_bytes, micro_batches=m)
    return cf.Workload(w.name, w.layers, w.mesh, net, S=w.S, seed=w.seed)


@pytest.mark.parametrize("m", [0, 1, 4, 100])
@pytest.mark.parametrize("which", ["tiny", "transformer24", "k6", "k216", "fused"])
def test_accumulation(adl, which, m):
    if which == "tiny":
        w = cf.config1_tiny()
    elif which == "transformer24":
        w = cf.config3_transformer24()
        w = cf.Workload(w.name, w.layers[:, :25], w.mesh, w.net, S=8)
    elif which == "k6":
        b = cf.config4_batched(Bp=3, L=6, seed=1)
        w = cf.Workload("k6", b.layers, cf.Mesh((8,), (1,)), b.net, S=2)
    elif which == "k216":
        w = cf.config5_transformer96()
        w = cf.Workload(w.name, w.layers[:, :10], w.mesh, w.net, S=4)
    else:
        w = cf.config4_batched(Bp=320, L=6, seed=2)
    w = _with_m(w, m)
    init = w.cd_init()
    n = min(w.Bp, 12)
    ws = cf.Workload(w.name, np.ascontiguousarray(w.layers[:n]), w.mesh, w.net, S=w.S, seed=w.seed)
    oT, onode, omask = ref.build_tables(ws.layers, ref.mesh_of(ws), ref.net_of(ws))
    odc, ods = ref.chain_dp(oT)
    occ, ocs, osw = ref.coord_descent(oT, np.ascontiguousarray(init[:n]), w.max_sweeps)
    d_layers = adl.layers_to_device(w.layers)
    one = adl.search(d_layers, w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=w.max_sweeps, want_node_mask=True)
    T, node, mask = adl.build_tables(d_layers, w.mesh, w.net)
    torch.cuda.synchronize()
    assert torch.equal(one["T"], T) and torch.equal(one["node"], node) and torch.equal(one["mask"], mask)
    for name, g, o in (("T", T, oT), ("node", node, onode), ("mask", mask, omask), ("dp_cost", one["opt_cost"], odc),
                       ("dp_strategy", one["strategy"], ods), ("cd_cost", one["cd_cost"], occ), ("cd_strategy", one["cd_strategy"], ocs),
                       ("cd_sweeps", one["cd_sweeps"], osw)):
        assert np.array_equal(g[:n].cpu().numpy(), o), name
