"""Multi-GPU plumbing: replicas only.

Events are independent, a PU200 event is ~2 MB of input and ~40 us of B200 time, so the path does
not shard inside an event: every rank (one process per GPU) runs the whole chain on its own events.
There is no collective on the data path; ``torch.distributed`` only agrees on which events a rank
takes and reduces the timings (max over ranks) and counters (sum over ranks) for reporting.
"""
from __future__ import annotations


def event_indices(rank: int, world: int, n_batches: int, events_per_batch: int) -> list[list[int]]:
    """Event numbers (the ``index`` of lst_inputs.make_config_event("C5", ...)) of every batch of
    ``rank``: contiguous blocks, disjoint across ranks, identical for a given (rank, world)."""
    if not (0 <= rank < world) or n_batches < 0 or events_per_batch <= 0:
        raise ValueError("bad replica layout")
    first = rank * n_batches * events_per_batch
    return [list(range(first + b * events_per_batch, first + (b + 1) * events_per_batch)) for b in range(n_batches)]


def _reduce(values, op_name: str, device):
    import torch
    import torch.distributed as dist

    vals = [float(v) for v in values]
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return vals
    t = torch.tensor(vals, dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return [float(v) for v in t.cpu()]


def max_over_ranks(values, device=None) -> list[float]:
    """Element-wise maximum over all ranks (device times of a timed region: the slowest rank counts)."""
    return _reduce(values, "MAX", device)


def sum_over_ranks(values, device=None) -> list[float]:
    """Element-wise sum over all ranks (events, objects, launches)."""
    return _reduce(values, "SUM", device)


def barrier() -> None:
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
