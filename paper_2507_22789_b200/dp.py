"""Data-parallel plumbing for the scoring path: whole groups per rank, W replicated
("use all GPUs for training and rollout log probability calculations"; DP at
PAPER.md:86).  Scoring (stage 3) needs no data-path collective: ranks only agree on timing and
token counts.  Training (stage 4) across ranks needs exactly two exchanges: the
global scored-token count before the backward, and an all-reduce of dW (and of the loss scalars)
after it -- `global_grad_scale` and `all_reduce_mean` below.  dH stays local (each rank owns its
tokens); like dW before the mean it is world x the global gradient, which the trunk's own
gradient averaging over ranks divides out.  Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
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


def global_grad_scale(n_scored_local: float) -> float:
    """`grad_loss` to pass to gc_grpo_loss_bwd on this rank so that the MEAN over ranks of the
    local dW (and of the local loss) is the gradient (loss) of the global token-mean objective
    sum_all m l / sum_all m:  local dW_r = grad_loss_r / n_r * S_r with S_r the rank's un-normalised
    sum, so grad_loss_r = world * n_r / N makes mean_r dW_r = (1/N) sum_r S_r.  One all-reduce of a
    scalar.  (Equal per-rank counts give 1.0.)"""
    if not is_dist():
        return 1.0
    n = torch.tensor([float(n_scored_local)], dtype=torch.float64, device=_device())
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    total = float(n.item())
    return dist.get_world_size() * float(n_scored_local) / total if total > 0 else 0.0


def all_reduce_mean(*tensors: torch.Tensor) -> None:
    """In-place mean over ranks (dW [V,D] fp32: 2-8 GB, NCCL over NVLink on GPUs; loss scalars)."""
    if not is_dist():
        return
    w = dist.get_world_size()
    for t in tensors:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        t.div_(w)


def shard_rows_for(V: int, world: int) -> int:
    """Rows per dW shard: ceil(V / world) rounded up to a multiple of 32 (a warp's slab of the dW
    epilogue must not straddle two owners)."""
    return -(-(-(-V // world)) // 32) * 32


def exchange_dw_shards(shard: torch.Tensor):
    """Every rank passes its own fp32 dW shard [shard_rows, D] (CUDA); returns (ptrs, keepalive):
    ptrs[r] = device address of rank r's shard as seen from this process -- its own tensor, or the
    peer's memory opened through CUDA IPC (same node; NVLink / NVSwitch carries the traffic when the
    peer is another GPU, for which peer access is switched on by a first device-to-device copy).
    `keepalive` must outlive every kernel that uses the pointers.  Collective over the default
    group (any backend: only picklable IPC handles travel through it)."""
    from torch.multiprocessing.reductions import reduce_tensor
    assert shard.is_cuda and shard.dtype == torch.float32 and shard.is_contiguous()
    if not is_dist():
        return [shard.data_ptr()], [shard]
    rank, world = dist.get_rank(), dist.get_world_size()
    gathered = [None] * world
    dist.all_gather_object(gathered, reduce_tensor(shard))
    tensors = []
    for r, (rebuild, args) in enumerate(gathered):
        if r == rank:
            tensors.append(shard)
            continue
        t = rebuild(*args)
        if t.device != shard.device:
            _ = t[:1].to(shard.device)          # first peer copy enables peer access in torch
        tensors.append(t)
    return [t.data_ptr() for t in tensors], tensors
