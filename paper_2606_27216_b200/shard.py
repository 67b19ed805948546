"""Multi-GPU sharding of the HiMuon step: whole matrices per rank, no data-path collective.

Tiles are independent units (with bank-sharded parameters "the tiled Newton-Schulz
computation is rank-local and does not require an optimizer-internal all-gather"), so a parameter set is split
across ranks by whole matrices; every rank builds its own himuon_plan over its share.  Host logic only."""
from __future__ import annotations

from typing import List, Sequence


def shard_layers(n_elements: Sequence[int], world: int) -> List[List[int]]:
    """Balanced split of layer indices over `world` ranks: largest matrix first onto the lightest rank
    (deterministic: ties go to the lower rank, equal sizes keep their order)."""
    if world < 1:
        raise ValueError("world must be >= 1")
    loads = [0] * world
    out: List[List[int]] = [[] for _ in range(world)]
    for i in sorted(range(len(n_elements)), key=lambda k: (-int(n_elements[k]), k)):
        r = min(range(world), key=lambda k: (loads[k], k))
        out[r].append(i)
        loads[r] += int(n_elements[i])
    for r in range(world):
        out[r].sort()
    return out


def max_over_ranks(value: float, device=None) -> float:
    """max of a per-rank scalar (e.g. the device-timed ms of the step) over the default process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
