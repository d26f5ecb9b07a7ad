"""Multi-GPU plumbing of the hot path: every (b,h) is an independent unit through all steps, so the path
shards over contiguous head ranges with NO data-path collective; torch.distributed is used only to agree on timings
(max over ranks) and to gather per-rank results.  Pure host logic: works on the gloo backend without a GPU."""
from __future__ import annotations

import numpy as np


def shard_heads(n_units: int, world_size: int, rank: int) -> np.ndarray:
    """Contiguous, balanced range of (b,h) unit indices owned by `rank` (int32, suitable as `head_sel`)."""
    if not (0 <= rank < world_size) or n_units < 0:
        raise ValueError('bad rank / world_size')
    base, rem = divmod(n_units, world_size)
    lo = rank * base + min(rank, rem)
    hi = lo + base + (1 if rank < rem else 0)
    return np.arange(lo, hi, dtype=np.int32)


def max_over_ranks(value: float, device='cpu') -> float:
    """Device time of a multi-GPU step = max over ranks (never wall clock)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_done_local: float, ms_local: float, device='cpu') -> float:
    """Whole-job throughput = units processed by all ranks / max-over-ranks time (units per second)."""
    import torch
    import torch.distributed as dist
    ms = max_over_ranks(ms_local, device)
    total = float(units_done_local)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([total], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        total = float(t.item())
    return total / (ms * 1e-3)
