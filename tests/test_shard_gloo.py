"""-m "not gpu": the N > 1 path (shard over noise sources, one gather of the loops) with world_size 2 on gloo."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1309_2256_b200 import shard


@pytest.mark.parametrize("n,nrhs,world", [(200, 12, 1), (200, 12, 2), (200, 12, 8), (5, 12, 4), (0, 12, 2), (24, 12, 2), (25, 4, 3)])
def test_source_batches_partition(n, nrhs, world):
    seen = []
    nb = []
    for r in range(world):
        b = shard.source_batches(n, nrhs, r, world)
        nb.append(len(b))
        for first, count in b:
            assert 1 <= count <= nrhs and first % nrhs == 0
            seen += list(range(first, first + count))
        assert shard.owned_sources(n, nrhs, r, world) == [f + k for f, c in b for k in range(c)]
    assert sorted(seen) == list(range(n))          # every source exactly once
    assert max(nb) - min(nb) <= 1                  # whole batches, balanced


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n, nrhs, T, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ids = shard.owned_sources(n, nrhs, rank, world)
    # stand-in for the loops of source r: a pattern that encodes r, n and t
    local = torch.zeros((len(ids), 16, T, 2), dtype=torch.float64)
    for k, r in enumerate(ids):
        local[k] = r + torch.arange(16 * T * 2, dtype=torch.float64).reshape(16, T, 2) / 1000.0
    full = shard.gather_loops(local, n, nrhs)
    ok = full.shape == (n, 16, T, 2)
    for r in range(n):
        ok = ok and torch.equal(full[r], r + torch.arange(16 * T * 2, dtype=torch.float64).reshape(16, T, 2) / 1000.0)
    q.put((rank, bool(ok)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("n,nrhs", [(29, 4), (8, 12), (50, 12)])
def test_gather_loops_world2_gloo(n, nrhs):
    world, T = 2, 6
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, nrhs, T, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True), (1, True)]


def test_gather_loops_single_process():
    local = torch.arange(3 * 16 * 4 * 2, dtype=torch.float64).reshape(3, 16, 4, 2)
    assert torch.equal(shard.gather_loops(local, 3, 12), local)
