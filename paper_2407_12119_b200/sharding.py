"""Multi-GPU plumbing of the hot path: events are independent in every stage, so the path
shards by contiguous event ranges with no exchange step -- replicas only, no data-path collective (DESIGN.md
sec. 10).  What is left to agree on between ranks is which events each one takes and how the per-rank timings
and counts become one whole-job number; both live here so that bench.py and the world-size-2 gloo test share
them.  No method arithmetic."""
from __future__ import annotations


def rank_events(rank: int, world: int, events_per_gpu: int) -> tuple[int, int]:
    """(first_event, n_events) of the seeded event stream that `rank` processes: weak scaling, every rank takes
    its own `events_per_gpu` consecutive events, ranks in stream order, no overlap."""
    if not (0 <= rank < world) or events_per_gpu < 0:
        raise ValueError("rank_events: need 0 <= rank < world and events_per_gpu >= 0")
    return rank * events_per_gpu, events_per_gpu


def whole_job(ms: float, counts: list[float], dist=None, device="cpu"):
    """Max over ranks of the timed region and sums over ranks of the per-rank counts (events, hits, edges ...).
    With dist = None (one process) the inputs are returned unchanged."""
    if dist is None:
        return ms, [float(c) for c in counts]
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([float(x) for x in counts], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(x) for x in c.tolist()]
