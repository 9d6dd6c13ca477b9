"""N > 1 host logic on CPU: world_size-2 gloo, problems sharded over ranks, results gathered.  The compute on each
shard is stood in for by the oracle here (tests may call it); on GPUs it is the CUDA path (bench.py --gpus N)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2301_06813_b200 import configs as cf
from paper_2301_06813_b200.shard import best_of_starts, gather_rows, shard_range


def test_shard_range_partitions():
    for n in (0, 1, 5, 4096, 4099):
        for world in (1, 2, 3, 8):
            spans = [shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def test_best_of_starts_lowest_index():
    c = torch.tensor([[5, 3, 3, 9], [1, 1, 1, 1], [7, 8, 9, 6]])
    b, i = best_of_starts(c)
    assert b.tolist() == [3, 1, 6] and i.tolist() == [1, 0, 3]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, Bp, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import ref
    w = cf.config4_batched(Bp=Bp, L=9, seed=4)
    lo, hi = shard_range(Bp, rank, world)
    T, _, _ = ref.build_tables(w.layers[lo:hi], ref.mesh_of(w), ref.net_of(w))
    c, s = ref.chain_dp(T)
    cc, cs, sw = ref.coord_descent(T, w.cd_init()[lo:hi], w.max_sweeps)
    cost = gather_rows(torch.from_numpy(c), Bp)
    strat = gather_rows(torch.from_numpy(s), Bp)
    cdc = gather_rows(torch.from_numpy(cc), Bp)
    # timing rule of bench.py: max over ranks
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    assert t.item() == world
    if rank == 0:
        np.savez(os.path.join(out_dir, "gathered.npz"), cost=cost.numpy(), strat=strat.numpy(), cdc=cdc.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_rank_gloo_shard_and_gather(tmp_path):
    from oracle import ref
    Bp = 7                                         # ragged: 4 + 3
    mp.spawn(_worker, args=(2, _free_port(), Bp, str(tmp_path)), nprocs=2, join=True)
    got = np.load(tmp_path / "gathered.npz")
    w = cf.config4_batched(Bp=Bp, L=9, seed=4)
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    c, s = ref.chain_dp(T)
    cc, _, _ = ref.coord_descent(T, w.cd_init(), w.max_sweeps)
    assert np.array_equal(got["cost"], c) and np.array_equal(got["strat"], s) and np.array_equal(got["cdc"], cc)
