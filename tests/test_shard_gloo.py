"""N > 1 host logic on CPU: world_size 2 over gloo.  No data-path collective exists;
what is covered is the rank arithmetic bench.py uses: spaxel partition, replica seeds, max-over-ranks timing."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2604_23305_b200 import shard


def test_partition_is_contiguous_balanced_and_complete():
    assert [e - b for b, e in shard.partition_spaxels(61, 8)] == [8, 8, 8, 8, 8, 7, 7, 7]
    for n in (0, 1, 7, 37, 61):
        for w in (1, 2, 3, 8):
            parts = shard.partition_spaxels(n, w)
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(w - 1))
            sizes = [e - b for b, e in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.partition_spaxels(5, 0)


def test_single_process_reduction_is_identity():
    assert shard.max_over_ranks(3.5) == 3.5
    assert shard.aggregate_throughput(100.0, 4, 5, 1000.0) == 2000.0


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        b, e = shard.partition_spaxels(61, world)[rank]
        counts = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(counts, torch.tensor([e - b], dtype=torch.int64))
        dist.barrier()
        ms = shard.max_over_ranks(10.0 + 5.0 * rank, dist)           # rank 1 is the slow one
        q.put((rank, [int(c.item()) for c in counts], ms, shard.replica_seed(3, rank)))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [[31, 30], [31, 30]]               # every rank sees the whole partition
    assert [r[2] for r in res] == [15.0, 15.0]                       # max over ranks on both
    assert [r[3] for r in res] == [3, 1003]
    assert shard.aggregate_throughput(61 * 347 * 1000 / 2, 2, 1, 15.0) == pytest.approx(61 * 347 * 1000 / 0.015)
