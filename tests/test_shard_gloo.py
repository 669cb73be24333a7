"""N > 1 host logic on CPU: world_size 2 over gloo: the rank arithmetic bench.py uses -- spaxel
partition, shard workloads, replica seeds, max-over-ranks timing -- and the one data-path collective of the sharded
mode, the all-reduce of the common-mode partial sums of Eq. 25 (the per-rank partial sums are made by the oracle here:
there is no GPU; the CUDA kernels that make them are compared with the same oracle in tests/test_gpu_parity.py)."""
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


def _cm_case():
    import numpy as np
    rng = np.random.default_rng(9)
    n_t, n_s, n_c = 11, 7, 6
    arcsec = np.pi / 180 / 3600
    Tb = rng.uniform(5.0, 40.0, (n_t, n_s, n_c))
    eta_z = rng.uniform(0.4, 0.95, n_c)
    csc = rng.uniform(1.1, 1.5, (n_t, n_s))
    daz = np.array([0, 100, 250, -300, 0, 220, -150.0]) * arcsec
    de = np.array([0, 0, 0, 100, -260, 220, 150.0]) * arcsec
    return Tb, eta_z, csc, daz, de, 200 * arcsec


def _cm_worker(rank, world, port, q):
    """Each rank holds a spaxel sub-range, forms its partial common-mode sum (oracle arithmetic), the sums and counts are
    all-reduced, and every rank finishes Eq. 25 on its own slab."""
    import numpy as np
    from oracle import oracle as O
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        Tb, eta_z, csc, daz, de, r_out = _cm_case()
        b, e = shard.partition_spaxels(Tb.shape[1], world)[rank]
        S = (np.hypot(daz[b:e], de[b:e]) > r_out).astype(np.float64)
        eta = eta_z[None, None, :] ** csc[:, b:e, None]
        partial = torch.from_numpy((S[None, :, None] * Tb[:, b:e] / (1 - eta)).sum(axis=1))
        total, n_out = shard.common_mode_allreduce(partial, int(S.sum()), dist)
        out = Tb[:, b:e] / eta - (1 - eta) / (eta * n_out) * total.numpy()[:, None, :]
        q.put((rank, b, e, n_out, out))
    finally:
        dist.destroy_process_group()


def test_common_mode_allreduce_world_size_2_gloo():
    """Spaxel-sharded Eq. 25: two ranks, one SUM all-reduce over [t x chan]: equals the single-process oracle."""
    import numpy as np
    from oracle import oracle as O
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_cm_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=120) for _ in range(2)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    Tb, eta_z, csc, daz, de, r_out = _cm_case()
    ref, S, _ = O.common_mode_subtract(Tb, eta_z, csc, daz, de, r_out)
    assert [r[3] for r in res] == [int(S.sum())] * 2
    got = np.concatenate([r[4] for r in res], axis=1)
    np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-12)
    # identity without a process group
    t = torch.ones(2, 3)
    assert shard.common_mode_allreduce(t, 4)[1] == 4


def test_shard_workload_keeps_the_global_spaxel_index():
    import numpy as np
    from paper_2604_23305_b200 import workloads as W
    w = W.random_workload(2, n_spaxel=7, n_chan=5, pink_noise=True)
    parts = shard.partition_spaxels(w.n_spaxel, 3)
    ws = [shard.shard_workload(w, b, e) for b, e in parts]
    assert [x.spaxel_index_base for x in ws] == [0, 3, 5]
    assert np.array_equal(np.concatenate([x.daz_rad for x in ws]), w.daz_rad)
    assert np.array_equal(np.concatenate([x.pink_A for x in ws]), w.pink_A)
    assert sum(x.n_spaxel for x in ws) == 7


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
