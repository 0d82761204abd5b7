"""Replica bookkeeping for multi-GPU runs ("replicas only").

The split-step path does not shard (every transform is global), so N GPUs run N independent
simulations, one context per rank, with NO data-path collective.  The only communication is this
module's: a barrier around the timed region and a MAX over ranks of the device-measured times, so
that the whole-job figure is (units all ranks processed) / (slowest rank's time).  Works with any
torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import Sequence, Tuple


def rank_world() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when run directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def max_over_ranks(values: Sequence[float], device="cpu"):
    """Element-wise MAX of per-rank measurements over all ranks (identity when not initialised)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_rate(cells_per_rank: int, steps: int, world: int, slowest_ms: float) -> float:
    """cell-updates/s of the whole job: every rank advances its own replica `steps` steps."""
    return world * cells_per_rank * steps / (slowest_ms * 1e-3)
