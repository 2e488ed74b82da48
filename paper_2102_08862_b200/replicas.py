"""Multi-GPU use of the tracker: **replicas only** (DESIGN.md §9).

BASELINE.json L5 fixes "one GPU only" for the path; the paper's own multi-GPU use is independent time frames on
the 8 GPUs of a server.  So rank r tracks its own frame (seed + r) with no data-path collective,
and the only exchange is the reduction of the timing at the end: the job's time is the MAX over ranks, its work
the SUM of the clusters all ranks tracked.  This module holds that host logic (no tracker arithmetic), so that
``bench.py`` and the world_size-2 gloo test share it.
"""
from __future__ import annotations

import os
from typing import Tuple


def rank_world_local() -> Tuple[int, int, int]:
    """(RANK, WORLD_SIZE, LOCAL_RANK) as torchrun exports them; (0, 1, 0) in a plain ``python`` run."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def frame_seed(base_seed: int, rank: int) -> int:
    """Seed of the time frame rank ``rank`` generates: every replica tracks a different frame."""
    return int(base_seed) + int(rank)


def aggregate(total_ms: float, n_clusters: int, steps: int, world: int, device=None) -> Tuple[float, float, float]:
    """Whole-job numbers from this rank's timed region.

    total_ms    device time of this rank's ``steps`` timed steps (CUDA events)
    n_clusters  clusters this rank tracks per step
    Returns (ms_per_step, clusters_per_second, n_clusters_all_ranks) with ms_per_step = max over ranks / steps and
    clusters_per_second = sum over ranks of n_clusters / ms_per_step.  Every rank gets the same triple.
    ``world`` > 1 needs an initialised ``torch.distributed`` process group (nccl on GPUs, gloo in the CPU test).
    """
    if steps <= 0:
        raise ValueError("steps must be positive")
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            raise RuntimeError("aggregate(world > 1) needs an initialised process group")
        t_max = torch.tensor([float(total_ms)], dtype=torch.float64, device=device)
        n_sum = torch.tensor([float(n_clusters)], dtype=torch.float64, device=device)
        dist.all_reduce(t_max, op=dist.ReduceOp.MAX)
        dist.all_reduce(n_sum, op=dist.ReduceOp.SUM)
        total_ms_max, n_all = float(t_max[0]), float(n_sum[0])
    else:
        total_ms_max, n_all = float(total_ms), float(n_clusters)
    ms_per_step = total_ms_max / steps
    return ms_per_step, n_all / (ms_per_step * 1e-3), n_all


def max_over_ranks(value: float, world: int, device=None) -> float:
    """MAX over ranks of a scalar (per-step end-to-end time)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])
