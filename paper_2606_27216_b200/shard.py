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


def owner_of(parts: Sequence[Sequence[int]]) -> List[int]:
    """Inverse of `shard_layers`: owner rank of every layer index."""
    n = sum(len(p) for p in parts)
    own = [-1] * n
    for r, p in enumerate(parts):
        for i in p:
            if not 0 <= i < n or own[i] >= 0:
                raise ValueError("parts do not cover 0..n-1 exactly once")
            own[i] = r
    if any(o < 0 for o in own):
        raise ValueError("parts do not cover 0..n-1")
    return own


def exchange_updated_weights(Ws, parts: Sequence[Sequence[int]], group=None) -> int:
    """Replicated (DDP) parameter layout: every rank holds every W, the gradients arrive
    all-reduced, each rank runs the HiMuon step on ITS matrices only (its momentum shard stays with it), and
    the updated matrices are then sent from their owner to all ranks - the one exchange this layout needs
    per step, sum_l H_l W_l (n-1)/n elements received per rank.  All broadcasts are issued asynchronously
    and waited on together, so NCCL overlaps them over NVLink; in-place into the parameter tensors, no
    staging copy.  (With parameters already sharded by whole matrices - the paper's bank-sharded FSDP
    layout, PAPER.md:237 - there is nothing to exchange and this is not called.)  Returns the number of
    bytes this rank received."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return 0
    world = dist.get_world_size(group)
    if world == 1:
        return 0
    if len(parts) != world:
        raise ValueError("one part per rank expected")
    rank = dist.get_rank(group)
    own = owner_of(parts)
    if len(own) != len(Ws):
        raise ValueError("parts and Ws disagree on the number of layers")
    works, received = [], 0
    for i, W in enumerate(Ws):
        if not W.is_contiguous():
            raise ValueError("broadcast in place needs contiguous parameter tensors")
        src = own[i] if group is None else dist.get_global_rank(group, own[i])
        works.append(dist.broadcast(W, src=src, group=group, async_op=True))
        if own[i] != rank:
            received += W.numel() * W.element_size()
    for w in works:
        w.wait()
    return received
