"""N > 1 path on CPU: two gloo ranks split the maps of a batch, the union covers every map exactly once, and the
max-over-ranks timing reduction used by bench.py works."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1104_0672_b200.sharding import shard_range


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, total, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = torch.zeros(total, dtype=torch.int64)
    for k in shard_range(total, world, rank):
        mine[k] = 1
    dist.all_reduce(mine)
    t = torch.tensor([1.0 + rank], dtype=torch.float64)          # "ms" of this rank
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.barrier()
    if rank == 0:
        q.put((mine.tolist(), float(t.item())))
    dist.destroy_process_group()


@pytest.mark.parametrize("total", [16, 5])
def test_two_rank_map_sharding(total):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, total, q)) for r in range(2)]
    for p in procs:
        p.start()
    cover, tmax = q.get(timeout=120)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert cover == [1] * total and tmax == 2.0


def test_shard_range_properties():
    for total in (0, 1, 7, 16):
        for world in (1, 2, 3, 8):
            parts = [list(shard_range(total, world, r)) for r in range(world)]
            assert sum(parts, []) == list(range(total))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)
