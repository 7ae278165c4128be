"""Host-side plumbing of the multi-GPU launch.

Environments are independent, so the path shards by env with NO data-path collective:
every rank owns a contiguous block of envs, its own context, its own event stream.  The only collectives
are the two bookkeeping reductions of the benchmark: max over ranks of the device time and sums of the
counters.  Nothing here touches the method's arithmetic.
"""
from __future__ import annotations

from typing import Sequence, Tuple

import torch
import torch.distributed as dist


def env_block(rank: int, world: int, num_envs: int) -> Tuple[int, int]:
    """Contiguous block [e0, e1) of the `num_envs` environments owned by `rank` of `world` ranks; block
    sizes differ by at most one, the first `num_envs % world` ranks take the larger ones."""
    if not (0 <= rank < world) or num_envs < 0:
        raise ValueError("need 0 <= rank < world and num_envs >= 0")
    q, r = divmod(num_envs, world)
    e0 = rank * q + min(rank, r)
    return e0, e0 + q + (1 if rank < r else 0)


def rank_seed(base_seed: int, rank: int) -> int:
    """Weak scaling: every rank runs a batch of the same shape with its own seed."""
    return base_seed + 1000 * rank


def reduce_max_sum(values_max: Sequence[float], values_sum: Sequence[float], device) -> Tuple[list, list]:
    """(max over ranks of `values_max`, sum over ranks of `values_sum`); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values_max], [float(v) for v in values_sum]
    a = torch.tensor(list(values_max), dtype=torch.float64, device=device)
    b = torch.tensor(list(values_sum), dtype=torch.float64, device=device)
    dist.all_reduce(a, op=dist.ReduceOp.MAX)
    dist.all_reduce(b, op=dist.ReduceOp.SUM)
    return a.tolist(), b.tolist()
