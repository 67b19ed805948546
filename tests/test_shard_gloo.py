"""The N > 1 host path on CPU: world-size-2 gloo process group, whole-matrix sharding of a parameter set
(SURVEY.md 8(e)), max-over-ranks timing reduction as bench.py uses it.  No GPU needed."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import himuon_inputs as I
from paper_2606_27216_b200.shard import max_over_ranks, shard_layers


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
