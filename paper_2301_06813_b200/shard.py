"""Multi-GPU plumbing: problems (or Coordinate Descent starts) are independent, so ONE workload is
partitioned contiguously over the ranks with no collective in the data path, and one exchange of the small result
rows ends the step: an all-gather of (cost, strategy) rows, followed -- when the starts of a problem were split -- by
the best-of-starts reduction.  A single chain's DP does not shard: replicas only.

Host logic only (torch.distributed, any backend).  The compute on a shard and the best-of-starts reduction are
INJECTED callables: the CUDA path (binding.search / binding.best_of_starts) in bench.py and the GPU tests, the CPU
oracle in the gloo tests -- this module holds no arithmetic of the method and imports neither.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [lo, hi) of n units for `rank`; the first n % world ranks get one extra unit."""
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def _world() -> tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def gather_rows(local: torch.Tensor, n_total: int) -> torch.Tensor:
    """All-gather rows that were sharded with shard_range (ragged shards are padded to the largest one)."""
    rank, world = _world()
    if world == 1:
        return local
    biggest = (n_total + world - 1) // world
    pad = torch.zeros((biggest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    out = []
    for r, p in enumerate(parts):
        lo, hi = shard_range(n_total, r, world)
        out.append(p[: hi - lo])
    return torch.cat(out, dim=0)


class ShardedSearch:
    """One workload over all ranks of the default process group, results complete on every rank.

    layers [Bp, L] records, init [Bp, S, L] starts (or None).
    mode "problems": rank r searches problems shard_range(Bp, r, world) with all their starts.
    mode "starts":   every rank holds all problems and runs Coordinate Descent from starts shard_range(S, r, world) only
                     (the tables of a problem are then built on every rank: replicas of (a1) and (a2)).
    local_shard:     `layers` / `init` are ALREADY this rank's shard of a world-times larger workload (weak scaling:
                     every rank generates its own problems); mode "problems" only.
    The shard is cut once, here; run() may be called every step.  The only communication is the final all-gather of
    the result rows."""

    def __init__(self, layers: np.ndarray, init: np.ndarray | None, mode: str = "problems", local_shard: bool = False):
        self.rank, self.world = _world()
        self.mode, self.has_init = mode, init is not None
        if mode == "problems":
            if local_shard:
                self.n_total = layers.shape[0] * self.world
                self.layers, self.init = layers, init
            else:
                self.n_total = layers.shape[0]
                lo, hi = shard_range(self.n_total, self.rank, self.world)
                assert hi > lo, "more ranks than problems"
                self.layers = np.ascontiguousarray(layers[lo:hi])
                self.init = None if init is None else np.ascontiguousarray(init[lo:hi])
        elif mode == "starts":
            assert init is not None and not local_shard, "mode 'starts' shards the Coordinate Descent starts of one workload"
            self.n_total = init.shape[1]
            lo, hi = shard_range(self.n_total, self.rank, self.world)
            assert hi > lo, "more ranks than starts"
            self.layers, self.init = layers, np.ascontiguousarray(init[:, lo:hi])
        else:
            raise ValueError(mode)

    def run(self, compute, best_of_starts=None):
        """compute(layers_shard, init_shard) -> dict of tensors: opt_cost [n], strategy [n, L] and, with starts, cd_cost
        [n, s], cd_strategy [n, s, L], cd_sweeps [n, s].  best_of_starts(cd_cost [Bp, S]) -> (best_cost [Bp], best_start
        [Bp]): smallest cost, smallest start on ties."""
        res = compute(self.layers, self.init)
        out = {}
        if self.mode == "problems":
            for k in ("opt_cost", "strategy") + (("cd_cost", "cd_strategy", "cd_sweeps") if self.has_init else ()):
                out[k] = gather_rows(res[k], self.n_total)
        else:
            out["opt_cost"], out["strategy"] = res["opt_cost"], res["strategy"]     # replicas: identical on every rank
            for k in ("cd_cost", "cd_strategy", "cd_sweeps"):
                t = res[k].transpose(0, 1).contiguous()                              # starts first: rows to gather
                out[k] = gather_rows(t, self.n_total).transpose(0, 1).contiguous()
        if self.has_init and best_of_starts is not None:
            out["best_cost"], out["best_start"] = best_of_starts(out["cd_cost"])
        return out


def sharded_search(layers: np.ndarray, init: np.ndarray | None, compute, best_of_starts=None, mode: str = "problems"):
    """ShardedSearch(...).run(...) in one call (strong scaling of one workload)."""
    return ShardedSearch(layers, init, mode).run(compute, best_of_starts)
