"""Multi-GPU = replicas over disjoint event ranges ("events are independent").

There is no data-path collective: every rank reconstructs its own batch on its own GPU.  The only communication is
the measurement plumbing of bench.py (a barrier, the max of the per-rank step time, the sum of the events), kept here
so that it can be exercised with the gloo backend on CPU.
"""
from __future__ import annotations


def batch_index_of(rank: int) -> int:
    """Seed offset of a rank's synthetic batch (seed = base + 1000*config + batch_index)."""
    return int(rank)


def event_range_of(rank: int, world: int, n_events: int) -> tuple[int, int]:
    """Contiguous share [first, last) of rank `rank` when ONE batch of n_events is split over `world` ranks."""
    base, extra = divmod(int(n_events), int(world))
    first = rank * base + min(rank, extra)
    return first, first + base + (1 if rank < extra else 0)


class Reducer:
    """max / sum over ranks of a Python float; identity when torch.distributed is not initialised."""

    def __init__(self, device=None):
        import torch
        import torch.distributed as dist

        self._torch, self._dist, self._device = torch, dist if dist.is_available() and dist.is_initialized() else None, device

    def _reduce(self, v: float, op_name: str) -> float:
        if self._dist is None:
            return float(v)
        t = self._torch.tensor([v], dtype=self._torch.float64, device=self._device)
        self._dist.all_reduce(t, op=getattr(self._dist.ReduceOp, op_name))
        return float(t.item())

    def max(self, v: float) -> float:
        return self._reduce(v, "MAX")

    def sum(self, v: float) -> float:
        return self._reduce(v, "SUM")

    def barrier(self) -> None:
        if self._dist is not None:
            self._dist.barrier()


def whole_job_value(reducer: Reducer, events_this_rank: int, ms_per_step_this_rank: float) -> tuple[float, float]:
    """(events/s of the whole job, ms per step) = all events / the slowest rank's step time."""
    ms = reducer.max(ms_per_step_this_rank)
    total = reducer.sum(float(events_this_rank))
    return total / (ms * 1e-3), ms
