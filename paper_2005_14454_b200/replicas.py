"""Multi-GPU = replicas only: one periodic lattice lives in ONE GPU's HBM and the path
has no data-path collective.  With N GPUs, rank r evolves its own, independent lattice (the paper's own use of many
runs: ensembles of seeds per era).  This module is the host logic of that launch, torch.distributed
plumbing only: which seed a rank runs, and how per-rank device times and unit counts combine into the whole-job
figure (max over ranks of the time, sum over ranks of the work).  It works with any backend (nccl on GPUs, gloo in
the CPU tests) and holds none of the method's arithmetic.
"""
from __future__ import annotations

import os


def rank_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process per GPU); (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of the replica that `rank` evolves: distinct, deterministic, never 0."""
    if base_seed < 0 or rank < 0:
        raise ValueError("seed and rank must be non-negative")
    return int(base_seed) + int(rank) + (1 if base_seed + rank == 0 else 0)


def aggregate(ms_local: float, units_local: float, dist=None, device="cpu"):
    """Whole-job (elapsed_ms, units): elapsed = MAX over ranks, units = SUM over ranks.

    `dist` is torch.distributed (initialised) or None for a single process.  Every rank gets the same result."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local), float(units_local)
    import torch

    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(ms: float, units: float) -> float:
    """units per second from a device time in milliseconds."""
    if not ms > 0.0:
        raise ValueError("elapsed time must be positive")
    return units / (ms * 1e-3)
