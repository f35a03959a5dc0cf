"""Host-side logic of the multi-GPU arm: "replicas only".

The SW sweep of one lattice runs on one GPU; N GPUs run N independent lattices (one process per GPU, different
seeds -- the natural way to produce the paper's temperature scans and independent runs).
There is no data-path collective: the only exchange is the reduction of the timings for the report.
Nothing here touches CUDA, so the same code runs under gloo on CPU (tests/test_replicas.py).
"""
from __future__ import annotations

import torch


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s lattice: distinct per rank, rank 0 keeps the workload's own seed."""
    return (base_seed + 7919 * rank) & 0xFFFFFFFFFFFFFFFF


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise MAX over all ranks of a list of floats (the device time of a multi-GPU number is the slowest
    rank's).  `dist` = torch.distributed when initialised, else None (single process)."""
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_ns_per_flip(max_ms: float, steps: int, sites_per_replica: int, world: int) -> float:
    """ns per spin flip of the whole job: every rank flipped steps * sites spins in max_ms milliseconds."""
    return max_ms * 1e6 / (float(world) * steps * sites_per_replica)
