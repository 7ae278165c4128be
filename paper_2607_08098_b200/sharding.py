"""Host-side plumbing of the multi-GPU launch.

Environments are independent, so the path shards by env with NO data-path collective:
every rank owns a contiguous block of envs, its own context, its own event stream.  The only collectives
are the two bookkeeping reductions of the benchmark: max over ranks of the device time and sums of the
counters.  Nothing here touches the method's arithmetic.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np
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


def gather_counts(n_local: int, device) -> List[int]:
    """The one optional collective of the sharded path: all-gather of the ranks' event counts, e.g.
    to place every rank's stream in one concatenated buffer.  Identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [int(n_local)]
    mine = torch.tensor([int(n_local)], dtype=torch.int64, device=device)
    out = [torch.zeros_like(mine) for _ in range(dist.get_world_size())]
    dist.all_gather(out, mine)
    return [int(t.item()) for t in out]


class ShardedEvis:
    """ONE batch of `num_envs` environments over the ranks of the process group (strong scaling): rank r owns the
    contiguous envs ``env_block(r, world, num_envs)`` with its own context on its own GPU, its own carried state and its
    own event stream; there is no exchange step (the envs are batched for efficiency only).

    ``step`` takes the rank's SLICE of the keyframe (``[e0:e1]`` of the batch tensors); events carry LOCAL env indices,
    ``global_env`` maps them back.  Noise events (``ctx.set_noise``) are keyed by the env's index in the whole batch
    (``evis_set_env_offset``), so the shards draw what the single context would; a hot-pixel mask is the rank's slice.  ``rank`` / ``world`` default to the process group's (1 rank without one), so the same
    code runs under ``torchrun`` and in a single process; passing them explicitly builds one shard by hand.
    """

    def __init__(self, num_envs: int, height: int, width: int, substeps: int, c_pos: float, c_neg: float,
                 log_eps: float, keyframe_dt: float, *, rank: Optional[int] = None, world: Optional[int] = None,
                 device: Optional[int] = None, **kw):
        from . import binding
        grouped = dist.is_available() and dist.is_initialized()
        self.world = int(world if world is not None else (dist.get_world_size() if grouped else 1))
        self.rank = int(rank if rank is not None else (dist.get_rank() if grouped else 0))
        self.num_envs = int(num_envs)
        self.e0, self.e1 = env_block(self.rank, self.world, self.num_envs)
        if self.e1 == self.e0:
            raise ValueError(f"rank {self.rank} of {self.world} owns no environment of {num_envs}")
        if device is None:
            device = torch.cuda.current_device()
        self.device = torch.device("cuda", device)
        self.ctx = binding.Evis(self.e1 - self.e0, height, width, substeps, c_pos, c_neg, log_eps, keyframe_dt,
                                device=device, **kw)
        self.ctx.set_env_offset(self.e0)          # noise events are keyed by the env's index in the whole batch

    def local(self, batch_tensor: torch.Tensor) -> torch.Tensor:
        """This rank's slice of a tensor that holds the whole batch (env-major)."""
        return batch_tensor[self.e0:self.e1].contiguous()

    def step(self, rad, mv_bwd, depth, mv_fwd=None, **kw):
        return self.ctx.step(rad, mv_bwd, depth, mv_fwd=mv_fwd, **kw)

    def read_events(self, **kw) -> np.ndarray:
        return self.ctx.read_events(**kw)

    def global_env(self, events: np.ndarray) -> np.ndarray:
        """Env index of every event in the whole batch."""
        return events["env"].astype(np.int64) + self.e0

    def gather_counts(self, n_local: int) -> List[int]:
        return gather_counts(n_local, self.device)

    def destroy(self) -> None:
        self.ctx.destroy()
