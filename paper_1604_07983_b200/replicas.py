"""T-parallel replicas ("Multi-GPU"): time slices are independent,
so N ranks run the single-GPU library on disjoint slices with no collective on the data path.
This module holds the host logic bench.py uses under torchrun: which slices a rank owns, and the
max-over-ranks of the device timings (the only communication).  It has no CUDA dependency, so the
N > 1 path is covered by world_size-2 gloo tests on CPU (tests/test_replicas_cpu.py)."""
from __future__ import annotations


def rank_slices(rank: int, world: int, T: int, count: int | None = None) -> list[int]:
    """Slices t = rank, rank + world, ... (< T) owned by `rank`; `count` cycles through them
    (bench.py times a fixed number of steps per rank: weak scaling)."""
    if not (0 <= rank < world) or T < 1:
        raise ValueError("bad rank / world / T")
    own = list(range(rank, T, world)) or [rank % T]
    if count is None:
        return own
    return [own[i % len(own)] for i in range(count)]


def max_over_ranks(values: list[float], device=None) -> list[float]:
    """Element-wise maximum over the ranks of the default process group (identity for one process)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return list(values)
    t = torch.tensor(values, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def aggregate_throughput(steps_per_rank: int, world: int, max_ms: float) -> float:
    """Whole-job slices per second: every rank ran `steps_per_rank` slices in at most `max_ms`."""
    return world * steps_per_rank / (max_ms * 1e-3)
