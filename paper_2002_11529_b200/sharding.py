"""Event-level data parallelism across GPUs (events are independent).

Rank r of N owns a contiguous range of events of the same seeded stream and runs the unchanged
single-GPU path on it: geometry replicated, no collective on the data path, outputs stay sharded.
The only exchanges are the two scalar reductions of the timing protocol (max of the device time, sum of
the events), which work over NCCL (device tensors) and gloo (host tensors) alike.  No arithmetic of the
method lives here.
"""
from __future__ import annotations


def shard_event_range(rank: int, world: int, events_per_rank: int) -> tuple[int, int]:
    """[first, last) of the global event stream owned by `rank` (weak scaling: fixed work per rank)."""
    if not (0 <= rank < world) or events_per_rank < 0:
        raise ValueError(f"bad shard request rank={rank} world={world} events_per_rank={events_per_rank}")
    return rank * events_per_rank, (rank + 1) * events_per_rank


def split_events(n_events: int, world: int) -> list[tuple[int, int]]:
    """Strong-scaling split of a fixed batch: contiguous, balanced to within one event, covering [0, n)."""
    if world < 1 or n_events < 0:
        raise ValueError("bad split request")
    q, r = divmod(n_events, world)
    out, lo = [], 0
    for k in range(world):
        hi = lo + q + (1 if k < r else 0)
        out.append((lo, hi))
        lo = hi
    return out


def reduce_job(local_ms: float, local_events: int, device=None):
    """(max over ranks of the timed milliseconds, sum over ranks of the events processed).
    Single process (no initialised process group): returns the inputs."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_ms), float(local_events)
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=device)
    n = torch.tensor([float(local_events)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t.item()), float(n.item())
