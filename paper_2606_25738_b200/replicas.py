"""Multi-GPU plumbing of the replica mode (the path does not shard; N ranks run N
independent batches and no collective touches the data path).

Only two things are distributed: which seed a rank generates its batch from, and how the per-rank timings
and unit counts combine into the whole-job number (units of all ranks / max-over-ranks time).  Both are
plain functions so that the N > 1 logic is testable with the gloo backend on CPU.
"""
from __future__ import annotations


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of rank ``rank``'s synthetic batch: replicas must not all time the same bytes."""
    return int(base_seed) + int(rank)


def aggregate(ms_local: float, cells_local: float, pairs_local: float, dist=None, device="cpu"):
    """(max-over-ranks ms, total cells, total pairs).  ``dist`` = an initialised torch.distributed module or
    None for a single process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local), float(cells_local), float(pairs_local)
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([float(cells_local), float(pairs_local)], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), float(c[0].item()), float(c[1].item())


def whole_job_gcups(ms_max: float, cells_total: float, steps: int) -> float:
    """GCUPS of the whole job: all ranks' cells per step / max-over-ranks time per step."""
    return cells_total / (ms_max / steps * 1e-3) / 1e9
