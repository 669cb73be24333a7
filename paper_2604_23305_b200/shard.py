"""Host-side logic of the N > 1 path.

The signal chain shards with no data-path exchange: spaxels (and whole observations) are independent.  Two modes:
  * replicas (bench.py default): every rank simulates an independent observation; torch.distributed carries the
    barrier and the max-over-ranks reduction of the timing, nothing else;
  * spaxel shards (bench.py --shard spaxel): every rank holds a contiguous sub-range of the instrument's spaxels
    (gt_config.spaxel_index_base keeps the RNG counters global, so the shards reproduce the one-plan TOD bit for
    bit); the only cross-spaxel term of the paper, the common-mode sum of Eq. 25, is ONE all-reduce
    over [t x chan] of the per-rank partial sums that gt_common_mode_partial makes (`common_mode_allreduce`).
This module holds the rank arithmetic only; it is exercised on CPU with the gloo backend (world_size 2) in
tests/test_shard_gloo.py.
"""
from __future__ import annotations

from typing import List, Tuple


def partition_spaxels(n_spaxel: int, world_size: int) -> List[Tuple[int, int]]:
    """[begin, end) spaxel range of every rank: contiguous, sizes differ by at most one, larger shares first
    (61 spaxels over 8 ranks -> 8,8,8,8,8,7,7,7)."""
    if n_spaxel < 0 or world_size < 1:
        raise ValueError("n_spaxel >= 0 and world_size >= 1 required")
    base, extra = divmod(n_spaxel, world_size)
    out, b = [], 0
    for r in range(world_size):
        n = base + (1 if r < extra else 0)
        out.append((b, b + n))
        b += n
    return out


def shard_workload(w, begin: int, end: int):
    """The workload restricted to spaxels [begin, end): offsets, per-detector pink-noise levels, and the global index
    of its first spaxel (RNG counter word 1 stays the instrument's spaxel index)."""
    nc = w.n_chan
    kw = dict(daz_rad=w.daz_rad[begin:end], del_rad=w.del_rad[begin:end],
              spaxel_index_base=int(getattr(w, "spaxel_index_base", 0)) + begin)
    if w.pink_A is not None:
        kw.update(pink_A=w.pink_A[begin * nc:end * nc], pink_alpha=w.pink_alpha[begin * nc:end * nc])
    return w.replace(**kw)


def common_mode_allreduce(partial, n_out: int, dist=None):
    """Eq. 25's sum over ALL spaxels from the per-rank partial sums: SUM all-reduce of the [t x chan] tensor (in
    place) and of the per-rank count of off-source spaxels.  Identity without an initialised process group.
    Returns (total, n_out_total)."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return partial, int(n_out)
    import torch
    dist.all_reduce(partial, op=dist.ReduceOp.SUM)
    n = torch.tensor([int(n_out)], dtype=torch.int64, device=partial.device)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return partial, int(n.item())


def replica_seed(seed: int, rank: int) -> int:
    """Independent observation per rank (weak scaling): distinct Philox keys, same workload shape."""
    return int(seed) + 1000 * int(rank)


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX all-reduce of one timing value (ms); identity without an initialised process group."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, world_size: int, steps: int, total_ms: float) -> float:
    """Whole-job value: units all ranks processed / max-over-ranks time."""
    return world_size * units_per_rank * steps / (total_ms * 1e-3)
