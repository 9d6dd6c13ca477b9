"""Multi-GPU plumbing: problems (or CD starts) are independent, so they are partitioned
contiguously over ranks with no collective in the data path; one gather of the small result rows at the end.

Host logic only (torch.distributed, any backend); the compute on each shard is the CUDA path.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [lo, hi) of n units for `rank`; the first n % world ranks get one extra unit."""
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def gather_rows(local: torch.Tensor, n_total: int) -> torch.Tensor:
    """All-gather rows that were sharded with shard_range (ragged shards are padded to the largest one)."""
    if not dist.is_initialized() or dist.get_world_size() == 1:
        return local
    world = dist.get_world_size()
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


def best_of_starts(cost: torch.Tensor) -> tuple[torch.Tensor, torch.Tensor]:
    """Smallest cost, then smallest start index, per problem: cost [Bp, S] -> (best cost [Bp], start [Bp])."""
    best, idx = cost.min(dim=1)
    first = (cost == best[:, None]).to(torch.int64).argmax(dim=1)      # argmax returns the first maximum
    return best, first
