"""Replicas-only multi-GPU: events are independent, so rank r of a job simply owns a
disjoint block of event seeds and there is no data-path collective.  torch.distributed is used only
for the barrier and the max-over-ranks step time."""
from __future__ import annotations

BASE_SEED = 1000


def event_seeds(rank: int, world: int, events_per_rank: int, base: int = BASE_SEED) -> list[int]:
    """Seeds of the synthetic events rank `rank` of `world` processes (weak scaling: every rank has
    `events_per_rank` events; blocks are contiguous and disjoint)."""
    if not (0 <= rank < world) or events_per_rank < 0:
        raise ValueError("bad rank / world / events_per_rank")
    return [base + rank * events_per_rank + i for i in range(events_per_rank)]


def job_events_per_s(world: int, events_per_rank: int, steps: int, max_ms_over_ranks: float) -> float:
    """Whole-job throughput: all ranks' events over the slowest rank's time."""
    return world * events_per_rank * steps / (max_ms_over_ranks * 1e-3)


def max_over_ranks(ms: float, dist=None, device=None) -> float:
    """MAX all-reduce of a per-rank time (identity when not distributed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
