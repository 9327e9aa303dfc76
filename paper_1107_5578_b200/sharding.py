"""Host-side logic of the N > 1 paths.  No field arithmetic here.

* A single propagation / GS loop does not shard: `bench.py --gpus N` runs N
  replicas, and the only inter-rank steps are a barrier and the max-over-ranks of the device time
  (`max_over_ranks`).
* `cwo_propagate_stack` shards by plane: rank r propagates the contiguous slice
  `plane_shard(n, world, r)` of `zs` (the planes of a 3-D diffraction are independent 2-D
  diffractions); u1 is replicated, the output stays sharded by plane, no data-path collective.
"""
from __future__ import annotations

from typing import Sequence, Tuple


def plane_shard(n: int, world: int, rank: int) -> Tuple[int, int]:
    """[start, stop) of the planes rank `rank` owns: contiguous, sizes differ by at most one,
    lower ranks take the remainder.  Empty when n < world and rank >= n."""
    if n < 0 or world <= 0 or not (0 <= rank < world):
        raise ValueError("plane_shard(n=%d, world=%d, rank=%d)" % (n, world, rank))
    base, rem = divmod(n, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def shard_zs(zs: Sequence[float], world: int, rank: int):
    a, b = plane_shard(len(zs), world, rank)
    return list(zs[a:b]), a


def max_over_ranks(ms: float, device=None) -> float:
    """Max of a per-rank device time over the default process group (identity when not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: Sequence[int], ms_max: float) -> float:
    """Units all ranks processed / the slowest rank's time."""
    return float(sum(units_per_rank)) / (ms_max * 1e-3)
