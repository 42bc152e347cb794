"""Timing plumbing of the multi-GPU benchmark: rank environment, MAX over ranks of the device time, whole-job GLUPS.

The lattice itself is split over the ranks as x-slabs by ``slab.py`` (``bench.py --gpus N``);
``bench.py --replicas`` instead runs N independent lattices, one per rank, with no data-path communication.  Either way
the only thing this module does is aggregate the timing -- barrier, MAX over ranks of the device time.  It works on any
``torch.distributed`` backend (nccl on the GPU box, gloo in the CPU tests) and holds none of the method's arithmetic.
"""
from __future__ import annotations

import os


def env_world():
    """(world_size, rank, local_rank) from the torchrun environment; (1, 0, 0) without it."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX of a per-rank scalar over all ranks (the value itself when not distributed)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    """SUM of a per-rank scalar over all ranks (site updates done by the whole job)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_glups(site_updates_local: float, ms_local: float, device="cpu"):
    """Whole-job throughput of independent replicas: all ranks' site updates divided by the slowest
    rank's device time.  Returns (GLUPS, ms_max)."""
    ms_max = max_over_ranks(ms_local, device)
    total = sum_over_ranks(site_updates_local, device)
    return total / (ms_max * 1e-3) / 1e9, ms_max
