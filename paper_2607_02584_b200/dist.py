"""Multi-GPU plumbing of the hot path: every (b,h) is an independent unit through all steps, so the path
shards over contiguous head ranges with NO data-path collective; torch.distributed is used only to agree on timings
(max over ranks) and to gather per-rank results.  Pure host logic: works on the gloo backend without a GPU."""
from __future__ import annotations

import os
import socket
import subprocess
import sys

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


# ---- starting the ranks ------------------------------------------------------------------------------------------------
def needs_relaunch(n_gpus: int, env=None) -> bool:
    """`--gpus N` with N > 1 in a process that no launcher started (no WORLD_SIZE in the environment): the caller has to
    start the N ranks itself.  Under torchrun (WORLD_SIZE set) the answer is False and the process is one of the ranks."""
    env = os.environ if env is None else env
    return n_gpus > 1 and 'WORLD_SIZE' not in env


def torchrun_argv(n_gpus: int, script: str, script_args, port: int | None = None) -> list:
    """The launch line of the bench contract: one process per GPU on this node, rendezvous on 127.0.0.1."""
    if port is None:
        with socket.socket() as sk:
            sk.bind(('127.0.0.1', 0))
            port = sk.getsockname()[1]
    return [sys.executable, '-m', 'torch.distributed.run', '--nnodes=1', '--nproc-per-node', str(n_gpus),
            '--master-addr', '127.0.0.1', '--master-port', str(port), script] + list(script_args)


def relaunch_under_torchrun(n_gpus: int, script: str, script_args, env=None) -> int:
    """Run `script` as n_gpus ranks and return the launcher's exit code (rank 0 prints the result line; the ranks'
    stdout / stderr pass through).  NCCL's communicator log stays on so that the number of ranks can be read from it."""
    env = dict(os.environ if env is None else env)
    env.setdefault('NCCL_DEBUG', 'INFO')
    env.setdefault('NCCL_DEBUG_SUBSYS', 'INIT')
    return subprocess.call(torchrun_argv(n_gpus, script, script_args), env=env)
