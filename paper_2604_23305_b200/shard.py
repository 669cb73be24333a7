"""Host-side logic of the N > 1 path.

The path shards with no data-path exchange: spaxels (and whole observations) are independent until the
data-reduction step Eq. 25, which is out of scope.  This module only holds the rank arithmetic
that `bench.py` uses under torchrun; it is exercised on CPU with the gloo backend (world_size 2) in
tests/test_shard_gloo.py.  There is no collective on the data path: `torch.distributed` carries the barrier and
the max-over-ranks reduction of the timing, nothing else.
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
