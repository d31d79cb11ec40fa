"""Data-parallel plumbing for the scoring path: whole groups per rank, W replicated
("use all GPUs for training and rollout log probability calculations"; DP at
PAPER.md:86).  No data-path collective: ranks only agree on timing and token counts.
Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import os
from typing import Tuple

import torch
import torch.distributed as dist


def shard_groups(n_groups: int, world: int, rank: int) -> range:
    """Contiguous, balanced split of group indices: the first n_groups % world ranks get one more."""
    base, extra = divmod(n_groups, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def env_rank_world() -> Tuple[int, int, int]:
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def is_dist() -> bool:
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def _device():
    return torch.device("cuda", torch.cuda.current_device()) \
        if dist.get_backend() == "nccl" else torch.device("cpu")


def barrier():
    if is_dist():
        dist.barrier()


def reduce_step_stats(elapsed_ms: float, units: float) -> Tuple[float, float]:
    """(max over ranks of the device time, sum over ranks of the units processed)."""
    if not is_dist():
        return float(elapsed_ms), float(units)
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=_device())
    u = torch.tensor([units], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())
