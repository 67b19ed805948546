"""The N > 1 host path on CPU: world-size-2 gloo process group, whole-matrix sharding of a parameter set
(SURVEY.md 8(e)), max-over-ranks timing reduction as bench.py uses it.  No GPU needed."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import himuon_inputs as I
from paper_2606_27216_b200.shard import exchange_updated_weights, max_over_ranks, owner_of, shard_layers


def test_shard_layers_balanced_and_disjoint():
    spec = I.llama3_8b_spec()
    sizes = [l.H * l.W for l in spec.layers]
    for world in (1, 2, 4, 8):
        parts = shard_layers(sizes, world)
        flat = sorted(i for p in parts for i in p)
        assert flat == list(range(len(sizes))), "every layer exactly once"
        loads = [sum(sizes[i] for i in p) for p in parts]
        assert max(loads) - min(loads) <= max(sizes), "balanced to within one matrix"
    assert shard_layers([5, 5, 5], 2) == [[0, 2], [1]]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    spec = I.gpt2_small_spec()
    sizes = [l.H * l.W for l in spec.layers]
    mine = shard_layers(sizes, world)[rank]
    # every rank works on its own matrices only; the aggregate is assembled from per-rank element counts
    n_local = torch.tensor([sum(sizes[i] for i in mine)], dtype=torch.int64)
    dist.all_reduce(n_local)                       # bookkeeping only (not on the data path)
    ms = max_over_ranks(10.0 + rank)               # slowest rank defines the step time
    dist.barrier()
    q.put((rank, mine, int(n_local.item()), ms))
    dist.destroy_process_group()


def test_world_size_2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    spec = I.gpt2_small_spec()
    assert sorted(res[0][1] + res[1][1]) == list(range(len(spec.layers)))
    assert not set(res[0][1]) & set(res[1][1])
    assert res[0][2] == res[1][2] == spec.n_elements
    assert res[0][3] == res[1][3] == 11.0


def _worker_exchange(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    shapes = [(8, 12), (16, 4), (5, 7), (32, 32), (3, 9)]
    parts = shard_layers([h * w for h, w in shapes], world)
    # replicated layout: every rank starts from the same W; only the owner "steps" a matrix
    # (a stand-in update: the product path needs a GPU; the exchange does not care what the update was)
    Ws = [torch.full(s, float(i), dtype=torch.bfloat16) for i, s in enumerate(shapes)]
    for i in parts[rank]:
        Ws[i] += 100.0 * (rank + 1)
    got = exchange_updated_weights(Ws, parts)
    q.put((rank, [float(W[0, 0]) for W in Ws], [bool((W == W[0, 0]).all()) for W in Ws], got, parts))
    dist.destroy_process_group()


def test_exchange_updated_weights_world_size_2_gloo():
    """DDP layout: after the exchange every rank holds the owner's updated copy of every matrix."""
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker_exchange, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    parts = res[0][4]
    own = owner_of(parts)
    shapes = [(8, 12), (16, 4), (5, 7), (32, 32), (3, 9)]
    want = [float(i) + 100.0 * (own[i] + 1) for i in range(len(shapes))]
    for rank, vals, uniform, got, _ in res:
        assert vals == want and all(uniform)
        assert got == sum(2 * h * w for i, (h, w) in enumerate(shapes) if own[i] != rank)


def test_owner_of_rejects_gaps():
    import pytest
    assert owner_of([[0, 2], [1]]) == [0, 1, 0]
    with pytest.raises(ValueError):
        owner_of([[0], [2]])
