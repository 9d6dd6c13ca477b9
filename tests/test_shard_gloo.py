"""N > 1 host logic on CPU: world_size-2 gloo.  The function under test is shard.sharded_search -- the SAME function
bench.py --gpus N calls -- with the compute callable injected: the oracle here (tests may call it), the CUDA path on
GPUs (tests/test_gpu_shard.py runs that callable against the unsharded oracle on one rank)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2301_06813_b200 import configs as cf
from paper_2301_06813_b200.shard import gather_rows, shard_range, sharded_search


def test_shard_range_partitions():
    for n in (0, 1, 5, 4096, 4099):
        for world in (1, 2, 3, 8):
            spans = [shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def test_oracle_best_of_starts_lowest_index():
    """the oracle's reduction against the definition (numpy argmin returns the first minimum)"""
    from oracle import ref
    c = np.array([[5, 3, 3, 9], [1, 1, 1, 1], [7, 8, 9, 6]], np.int64)
    b, i = ref.best_of_starts(c)
    assert b.tolist() == [3, 1, 6] and i.tolist() == [1, 0, 3]
    rng = np.random.default_rng(0)
    c = rng.integers(0, 5, size=(50, 37)).astype(np.int64)
    b, i = ref.best_of_starts(c)
    assert np.array_equal(i, c.argmin(axis=1)) and np.array_equal(b, c.min(axis=1))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def oracle_compute(w):
    """compute callable for sharded_search backed by the CPU oracle"""
    from oracle import ref

    def compute(layers, init):
        T, _, _ = ref.build_tables(layers, ref.mesh_of(w), ref.net_of(w))
        c, s = ref.chain_dp(T)
        out = {"opt_cost": torch.from_numpy(c), "strategy": torch.from_numpy(s)}
        if init is not None:
            cc, cs, sw = ref.coord_descent(T, init, w.max_sweeps)
            out.update(cd_cost=torch.from_numpy(cc), cd_strategy=torch.from_numpy(cs), cd_sweeps=torch.from_numpy(sw))
        return out

    def best(cost):
        b, i = ref.best_of_starts(cost.numpy())
        return torch.from_numpy(b), torch.from_numpy(i)

    return compute, best


def _workload(mode):
    if mode == "problems":
        return cf.config4_batched(Bp=7, L=9, seed=4)            # ragged: 4 + 3 problems
    w = cf.config4_batched(Bp=3, L=9, seed=4)
    return cf.Workload(w.name, w.layers, w.mesh, w.net, S=5, seed=4)   # ragged: 3 + 2 starts


def _worker(rank, world, port, mode, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = _workload(mode)
    compute, best = oracle_compute(w)
    out = sharded_search(w.layers, w.cd_init(), compute, best, mode=mode)
    # timing rule of bench.py: max over ranks
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    assert t.item() == world
    np.savez(os.path.join(out_dir, f"gathered_{rank}.npz"), **{k: v.numpy() for k, v in out.items()})
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(120)
@pytest.mark.parametrize("mode", ["problems", "starts"])
def test_two_rank_gloo_shard_and_gather(tmp_path, mode):
    from oracle import ref
    mp.spawn(_worker, args=(2, _free_port(), mode, str(tmp_path)), nprocs=2, join=True)
    w = _workload(mode)
    init = w.cd_init()
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    c, s = ref.chain_dp(T)
    cc, cs, sw = ref.coord_descent(T, init, w.max_sweeps)
    bc, bs = ref.best_of_starts(cc)
    want = dict(opt_cost=c, strategy=s, cd_cost=cc, cd_strategy=cs, cd_sweeps=sw, best_cost=bc, best_start=bs)
    for rank in range(2):                                        # complete and identical on every rank
        got = np.load(tmp_path / f"gathered_{rank}.npz")
        for k, v in want.items():
            assert np.array_equal(got[k], v), (mode, rank, k)


def test_single_rank_is_the_identity():
    w = _workload("problems")
    compute, best = oracle_compute(w)
    a = sharded_search(w.layers, w.cd_init(), compute, best, mode="problems")
    b = sharded_search(w.layers, w.cd_init(), compute, best, mode="starts")
    for k in a:
        assert torch.equal(a[k], b[k]), k
    assert torch.equal(gather_rows(a["opt_cost"], 7), a["opt_cost"])
