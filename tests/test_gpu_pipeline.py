"""Pipeline-stage enumeration on the GPU (R27) against the oracle, bit for bit: the whole triangle of segment
optima, the transfer vector, the partition value + cuts for both objectives, and the per-segment strategies, for
configs 3 and 5 at stage counts 1, 2, 4 (each on the sub-mesh with 1 / stages of the nodes) and on random tables."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref
from paper_2301_06813_b200 import configs as cf

pytestmark = pytest.mark.gpu
PEN = 1 << 50


@pytest.fixture(scope="module")
def adl():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_2301_06813_b200 import binding
    binding.lib()
    return binding


def _compare(adl, w, stages, objective, oT=None):
    dl = adl.layers_to_device(w.layers)
    T, node, mask = adl.build_tables(dl, w.mesh, w.net)
    out = adl.pipeline_stages(dl[0], T[0], node[0], mask[0], w.mesh, w.net, stages, objective)
    torch.cuda.synchronize()
    if oT is None:
        oT = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    T1, n1, m1 = oT[0][0], oT[1][0], oT[2][0]
    tri = ref.segment_optima(T1, n1, m1)
    xfer = ref.stage_transfer(w.layers[0], ref.mesh_of(w), ref.net_of(w))
    val, cuts = ref.pipeline_partition(tri, xfer, stages, objective)
    sc, st = ref.segment_strategies(T1, n1, m1, cuts)
    assert np.array_equal(out["tri"].cpu().numpy(), tri)
    assert np.array_equal(out["xfer"].cpu().numpy(), xfer)
    assert int(out["value"][0]) == val and np.array_equal(out["cuts"].cpu().numpy(), cuts)
    assert np.array_equal(out["seg_cost"].cpu().numpy(), sc) and np.array_equal(out["strategy"].cpu().numpy(), st)
    return oT


@pytest.mark.parametrize("stages", [1, 2, 4])
def test_config3_stages(adl, stages):
    w = cf.config3_transformer24()
    sub = cf.Workload(w.name, w.layers, cf.Mesh((w.mesh.size[0] // stages, w.mesh.size[1]), w.mesh.link), w.net, S=1)
    oT = None
    for objective in (0, 1):
        oT = _compare(adl, sub, stages, objective, oT)


@pytest.mark.parametrize("stages", [1, 2, 4])
def test_config5_stages(adl, stages):
    """K = 216, L = 480: 115,440 segments; the oracle needs a few seconds per stage count"""
    w = cf.config5_transformer96()
    sub = cf.Workload(w.name, w.layers, cf.Mesh((w.mesh.size[0] // stages,) + tuple(w.mesh.size[1:]), w.mesh.link), w.net, S=1)
    _compare(adl, sub, stages, 1)


@pytest.mark.parametrize("K,L", [(6, 1), (6, 17), (36, 33), (216, 19), (81, 9), (243, 5)])
def test_random_tables(adl, K, L):
    """caller-supplied tables with heavy ties and penalties; ragged blocks of starts (L not a multiple of 16); the
    mixed-radix spaces of four / five mesh levels (K = 81, 243)"""
    rng = np.random.default_rng(K + L)
    T = rng.integers(0, 5, size=(L, K, K)).astype(np.int64)
    node = rng.integers(0, 5, size=(L, K)).astype(np.int64)
    mask = (rng.random((L, K)) > 0.2).astype(np.uint8)
    T += node[:, None, :] + np.where(mask == 1, 0, PEN)[:, None, :]
    mesh = {6: cf.Mesh((2,), (1,)), 36: cf.Mesh((2, 2), (1, 0)), 216: cf.Mesh((2, 2, 2), (1, 1, 0)),
            81: cf.Mesh((2, 2, 2, 2), (1 | 0x700, 0x700, 0x700, 0x700)), 243: cf.Mesh((2,) * 5, (1 | 0x700,) + (0x700,) * 4)}[K]
    layers = cf.config4_batched(Bp=1, L=L, seed=3).layers
    w = cf.Workload("rand", layers, mesh, cf.Net(cf.ALPHA_PS, (3, 40), 0, micro_batches=3), S=1)
    dl = adl.layers_to_device(w.layers)
    tri = ref.segment_optima(T, node, mask)
    xfer = ref.stage_transfer(w.layers[0], ref.mesh_of(w), ref.net_of(w))
    for stages in sorted({1, min(2, L), min(3, L), L}):
        for objective in (0, 1):
            out = adl.pipeline_stages(dl[0], torch.from_numpy(T).cuda(), torch.from_numpy(node).cuda(), torch.from_numpy(mask).cuda(),
                                      w.mesh, w.net, stages, objective)
            val, cuts = ref.pipeline_partition(tri, xfer, stages, objective)
            sc, st = ref.segment_strategies(T, node, mask, cuts)
            assert np.array_equal(out["tri"].cpu().numpy(), tri) and np.array_equal(out["xfer"].cpu().numpy(), xfer)
            assert int(out["value"][0]) == val and np.array_equal(out["cuts"].cpu().numpy(), cuts)
            assert np.array_equal(out["seg_cost"].cpu().numpy(), sc) and np.array_equal(out["strategy"].cpu().numpy(), st)


def test_errors(adl):
    T = torch.zeros((3, 36, 36), dtype=torch.int64, device="cuda")
    node = torch.zeros((3, 36), dtype=torch.int64, device="cuda")
    mask = torch.ones((3, 36), dtype=torch.uint8, device="cuda")
    w = cf.config4_batched(Bp=1, L=3)
    dl = adl.layers_to_device(w.layers)
    with pytest.raises(adl.AutoddlError, match="stages"):
        adl.pipeline_stages(dl[0], T, node, mask, w.mesh, w.net, 4, 1)
    with pytest.raises(adl.AutoddlError, match="objective"):
        adl.pipeline_stages(dl[0], T, node, mask, w.mesh, w.net, 2, 7)
