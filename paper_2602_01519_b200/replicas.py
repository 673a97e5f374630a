"""N > 1: independent replicas, one process per GPU, no collective on the data path.

The link-stage path shards by request: a request's block table and attention depend on nothing
but the chunks it links, so rank r takes a contiguous slice of the request list and owns a pool holding those
chunks.  The only cross-rank step is the timing reduction of ``bench.py`` (max over ranks)."""
from __future__ import annotations

from typing import Tuple


def shard_range(num_requests: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous request slice [begin, end) of `rank`; sizes differ by at most one, earlier ranks take the extra."""
    if world <= 0 or not (0 <= rank < world) or num_requests < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(num_requests, world)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def max_over_ranks(x: float, device=None) -> float:
    """MAX all-reduce of one scalar over the default process group (identity when there is none)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
