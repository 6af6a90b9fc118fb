"""Multi-GPU plumbing of bench.py: walkers are independent, so N ranks each run
their own batch with no data-path collective; only the timing is combined (max over ranks) and
the accepted-move counts summed.  Works on any torch.distributed backend (nccl on the GPU box,
gloo in the CPU tests)."""
from __future__ import annotations


def rank_seed(config_seed: int, rank: int, batch: int) -> int:
    """First walker seed of `rank`: walker w of rank r uses seed config_seed + r*batch + w, so the
    ranks' walkers are disjoint and rank 0 reproduces the single-GPU run."""
    return int(config_seed) + int(rank) * int(batch)


def combine(ms: float, accepted: int, device=None):
    """-> (max over ranks of ms, sum over ranks of accepted).  No-op without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms), int(accepted)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    a = torch.tensor([int(accepted)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(a, op=dist.ReduceOp.SUM)
    return float(t.item()), int(a.item())


def moves_per_second(ms_total: float, steps: int, accepted_all_ranks_per_step: int) -> float:
    """Whole-job throughput: accepted moves of all ranks in one step / (max-over-ranks time per step)."""
    return accepted_all_ranks_per_step / (ms_total / steps * 1e-3)
