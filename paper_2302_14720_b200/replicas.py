"""Host-side logic of the multi-GPU run: the path runs on one GPU, so N GPUs are N
independent replicas -- one lattice per rank, distinct seeds, no data-path collective.  The only exchanges are
bench.py's barrier and the max-over-ranks of the device time.  Backend-agnostic (nccl on the GPU box, gloo in the
CPU tests); holds none of the method's arithmetic.
"""
from __future__ import annotations

BASE_SEED = 6          # BASELINE configs[3]


def replica_seed(rank: int, base: int = BASE_SEED) -> int:
    """Seed of the replica on `rank`: configs[3] uses seed 6; replicas take 6 + rank."""
    if rank < 0:
        raise ValueError("rank must be >= 0")
    return base + rank


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """All-reduce MAX of a scalar (the timed region's duration).  dist = torch.distributed or None (one rank)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(sites_per_rank: int, steps: int, world: int, ms_max: float) -> float:
    """Site-updates per second of the whole job: every rank sweeps its own lattice `steps` times within the
    slowest rank's `ms_max` milliseconds (weak scaling)."""
    if ms_max <= 0:
        raise ValueError("ms_max must be positive")
    return world * sites_per_rank * steps / (ms_max * 1e-3)
