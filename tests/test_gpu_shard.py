"""The sharded CUDA path on one rank: shard.sharded_search with the compute callable bench.py injects (binding.search on
the shard + the library's best-of-starts kernel) against the unsharded oracle; and the library reduction on its own."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref
from paper_2301_06813_b200 import configs as cf
from paper_2301_06813_b200.shard import shard_range, sharded_search

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def adl():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_2301_06813_b200 import binding
    binding.lib()
    return binding


def test_best_of_starts_kernel(adl):
    rng = np.random.default_rng(1)
    for Bp, S, hi in [(1, 1, 5), (3, 2, 2), (17, 33, 3), (300, 64, 4), (5, 1000, 10**12), (4096, 1, 7)]:
        c = rng.integers(0, hi, size=(Bp, S)).astype(np.int64)
        c[rng.random(c.shape) < 0.1] += 1 << 50
        b, i = adl.best_of_starts(torch.from_numpy(c).cuda())
        ob, oi = ref.best_of_starts(c)
        assert np.array_equal(b.cpu().numpy(), ob) and np.array_equal(i.cpu().numpy(), oi), (Bp, S)
    with pytest.raises(adl.AutoddlError):
        adl.best_of_starts(torch.zeros((2, 2), dtype=torch.int32, device="cuda"))      # wrong dtype is refused by the binding


@pytest.mark.parametrize("mode", ["problems", "starts"])
def test_sharded_search_cuda_compute(adl, mode):
    """every shard a 2- or 3-rank job would compute, run here one after the other through the CUDA callable, then
    assembled the way gather_rows does: equal to the unsharded oracle"""
    from bench import cuda_compute
    w = cf.config4_batched(Bp=601, L=12, seed=9)
    w = cf.Workload(w.name, w.layers, w.mesh, w.net, S=5, seed=9)
    init = w.cd_init()
    compute, best = cuda_compute(adl, w)
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    c, s = ref.chain_dp(T)
    cc, cs, sw = ref.coord_descent(T, init, w.max_sweeps)
    bc, bs = ref.best_of_starts(cc)
    # world = 1 through the function bench.py calls
    out = sharded_search(w.layers, init, compute, best, mode=mode)
    torch.cuda.synchronize()
    for k, v in dict(opt_cost=c, strategy=s, cd_cost=cc, cd_strategy=cs, cd_sweeps=sw, best_cost=bc, best_start=bs).items():
        assert np.array_equal(out[k].cpu().numpy(), v), k
    # the shards of a 3-rank job, computed one by one
    for world in (2, 3):
        parts = []
        for r in range(world):
            if mode == "problems":
                lo, hi = shard_range(w.Bp, r, world)
                parts.append(compute(np.ascontiguousarray(w.layers[lo:hi]), np.ascontiguousarray(init[lo:hi])))
            else:
                lo, hi = shard_range(w.S, r, world)
                parts.append(compute(w.layers, np.ascontiguousarray(init[:, lo:hi])))
        torch.cuda.synchronize()
        axis = 0 if mode == "problems" else 1
        assert np.array_equal(torch.cat([p["cd_cost"] for p in parts], dim=axis).cpu().numpy(), cc)
        assert np.array_equal(torch.cat([p["cd_strategy"] for p in parts], dim=axis).cpu().numpy(), cs)
        assert np.array_equal(torch.cat([p["cd_sweeps"] for p in parts], dim=axis).cpu().numpy(), sw)
        if mode == "problems":
            assert np.array_equal(torch.cat([p["opt_cost"] for p in parts]).cpu().numpy(), c)
            assert np.array_equal(torch.cat([p["strategy"] for p in parts]).cpu().numpy(), s)
        else:
            for p in parts:
                assert np.array_equal(p["opt_cost"].cpu().numpy(), c)
