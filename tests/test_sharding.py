"""Host logic of the N>1 path (replicas only, no data-path collective): event
sharding and whole-job aggregation of bench.py, exercised with a world-size-2 gloo group on CPU."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seeds = bench.shard_seeds(rank, world, 4)
    local_ms = 2.0 + rank           # rank 1 is the slow one

    def red_max(v):
        t = torch.tensor([v], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def red_sum(v):
        t = torch.tensor([v], dtype=torch.int64)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return int(t.item())

    value, ms = bench.aggregate(local_ms, len(seeds), world, red_max, red_sum)
    value2, _ = bench.aggregate(local_ms, len(seeds), world, red_max)     # count = per-rank x world
    gathered = [None] * world
    dist.all_gather_object(gathered, seeds)
    if rank == 0:
        q.put((value, ms, value2, gathered))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_and_aggregation():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    value, ms, value2, gathered = q.get()
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert ms == 3.0                                   # max over ranks
    assert value == 8 / 3.0e-3 and value2 == value     # all ranks' events / slowest rank's time
    flat = [s for g in gathered for s in g]
    assert len(set(flat)) == 8 and flat == list(range(100, 108))   # disjoint, contiguous shards


def test_single_rank_is_identity():
    import bench
    assert bench.shard_seeds(0, 1, 64) == list(range(100, 164))
    v, ms = bench.aggregate(2.0, 64, 1)
    assert ms == 2.0 and v == 32000.0
