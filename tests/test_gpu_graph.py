"""The one-call path under CUDA graph capture: autoddl_search allocates nothing and synchronises nothing, its fork / join
side streams are ordered by events, so a caller can capture it once and replay it (the launch-bound small configs drop
from ~50-80 us to ~20-40 us per call).  A replay must give what the eager call gives (which the parity tests hold to the
oracle), bit for bit; the allocation-free chain DP is captured the same way."""
import numpy as np
import pytest
import torch

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


def _capture(fn):
    g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            fn()
    return g


@pytest.mark.parametrize("k", [1, 3, 9])
def test_search_replays_from_a_graph(adl, k):
    """config 1: three kernels on one stream; config 3: class-space DP with the tables and the look-up CD on side streams;
    config 9: folded mesh, layer-parallel DP beside the look-up CD on the tables"""
    w = cf.CONFIGS[k]()
    init = w.cd_init()
    dl, dinit = adl.layers_to_device(w.layers), torch.from_numpy(init).cuda()
    work = torch.empty(adl.workspace_bytes(w.Bp, w.L, w.S, w.mesh), dtype=torch.uint8, device="cuda")
    out = adl.search(dl, w.mesh, w.net, init=dinit, max_sweeps=w.max_sweeps, work=work)       # eager (also creates the side streams)
    torch.cuda.synchronize()
    oT, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    want = dict(zip(("T", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps"),
                    (oT,) + ref.chain_dp(oT) + ref.coord_descent(oT, init, w.max_sweeps)))
    g = _capture(lambda: adl.search(dl, w.mesh, w.net, init=dinit, max_sweeps=w.max_sweeps, work=work, out=out))
    for rep in range(2):
        for v in out.values():
            if v is not None:
                v.fill_(-1 if v.dtype != torch.uint8 else 255)
        work.fill_(17 * rep)
        g.replay()
        torch.cuda.synchronize()
        for name, o in want.items():
            assert np.array_equal(out[name].cpu().numpy(), o), (k, rep, name)


def test_static_chain_dp_replays_from_a_graph(adl):
    mesh, K, Bp, L = cf.Mesh((4, 4), (cf.INTER, cf.INTRA)), 36, 2, 75
    T = np.random.default_rng(5).integers(0, 7, size=(Bp, L, K, K), dtype=np.int64)
    d_T = torch.from_numpy(T).cuda()
    out = (torch.empty(Bp, dtype=torch.int64, device="cuda"), torch.empty((Bp, L), dtype=torch.int32, device="cuda"))
    adl.chain_dp_static(d_T, mesh, out)                      # eager once: the symbol address is looked up outside the capture
    g = _capture(lambda: adl.chain_dp_static(d_T, mesh, out))
    out[0].fill_(-1); out[1].fill_(-1)
    g.replay()
    torch.cuda.synchronize()
    oc, os_ = ref.chain_dp(T)
    assert np.array_equal(out[0].cpu().numpy(), oc) and np.array_equal(out[1].cpu().numpy(), os_)
