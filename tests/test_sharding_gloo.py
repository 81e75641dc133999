"""N>1 host logic on CPU: contiguous spectrum shards cover the batch exactly once and the reported time is
the max over ranks (world_size 2, gloo backend, 127.0.0.1 rendezvous)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2512_24840_b200.sharding import max_over_ranks, shard_range


def test_shard_range_covers_batch_exactly_once():
    for B in (0, 1, 7, 64, 65536, 10_000_003):
        for world in (1, 2, 3, 8):
            spans = [shard_range(B, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == B
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def _worker(rank, world, port, B, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    a, b = shard_range(B, rank, world)
    mine = torch.zeros(B, dtype=torch.int32)
    mine[a:b] = 1                      # "fitted" spectra of this rank
    dist.all_reduce(mine)              # test-only collective: the data path itself has none
    t = max_over_ranks(1.0 + rank, dist)
    dist.barrier()
    q.put((rank, int(mine.min()), int(mine.max()), b - a, t))
    dist.destroy_process_group()


def test_two_ranks_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    B, world = 1001, 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, B, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert [r[3] for r in res] == [501, 500]
    assert all(r[1] == 1 and r[2] == 1 for r in res)      # every spectrum fitted exactly once
    assert all(r[4] == 2.0 for r in res)                   # max over ranks
