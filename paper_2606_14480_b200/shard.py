"""Event sharding over GPUs (events are independent, L392: the
farm is independent cards).  One process per GPU; rank r owns a contiguous event range; there is no
exchange step and no collective on the data path.  The only collectives are the reporting
reductions below (max of the device time, sums of the counters), which work on any
torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import Dict, Tuple


def event_range(rank: int, world: int, n_events: int) -> Tuple[int, int]:
    """Contiguous strong-scaling shard [start, stop) of n_events events for `rank` of `world`;
    the first n_events % world ranks take one event more."""
    if not (world >= 1 and 0 <= rank < world and n_events >= 0):
        raise ValueError(f"bad shard request rank={rank} world={world} n_events={n_events}")
    q, r = divmod(n_events, world)
    start = rank * q + min(rank, r)
    return start, start + q + (1 if rank < r else 0)


def weak_chunks(rank: int, events_per_rank: int, chunk: int = 1024) -> Tuple[int, int]:
    """Weak-scaling shard: rank r generates its own events_per_rank events from generator chunks
    [first, first + n): (first_chunk, n_chunks).  Chunk k is seeded by (seed, k), so ranks never
    share an event and a rank's batch does not depend on the world size."""
    if rank < 0 or events_per_rank < 0 or chunk <= 0:
        raise ValueError("bad weak shard request")
    n = (events_per_rank + chunk - 1) // chunk
    return rank * n, n


def reduce_report(total_ms: float, counters: Dict[str, int], device="cpu") -> Tuple[float, Dict[str, int]]:
    """(max over ranks of total_ms, sum over ranks of each counter).  Identity when torch.distributed
    is not initialised (single process)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(total_ms), {k: int(v) for k, v in counters.items()}
    t = torch.tensor([float(total_ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    keys = sorted(counters)
    c = torch.tensor([int(counters[k]) for k in keys], dtype=torch.int64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), {k: int(v) for k, v in zip(keys, c.tolist())}
