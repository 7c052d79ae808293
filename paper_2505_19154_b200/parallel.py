"""Multi-GPU plumbing of the FHGS hot path.

One process per GPU (`torch.distributed`, backend "nccl" on GPUs, "gloo" in the CPU tests).  The path
shards in two ways, and this module holds only the host-side logic of both -- no arithmetic of the method:

  * independent frames (what `bench.py --gpus N` times): every rank renders and fuses its own frame, no
    data-path collective; only the timing is reduced (`max_over_ranks`).
  * view-sharded multi-view fusion: the accumulators num[N,D], den[N] (the paper's "cumulative-weight
    buffers") are sums over views, so each rank fuses its share of the views
    (`shard_views`) into private accumulators and ONE all-reduce(sum) of num and den
    (`allreduce_accumulators`) precedes the finalise step.  That all-reduce is the only exchange step of
    the path.
"""
from __future__ import annotations

from typing import Callable, List, Sequence

import torch
import torch.distributed as dist


def world_info() -> tuple:
    """(rank, world_size) of the default process group, (0, 1) when torch.distributed is not initialised."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def shard_views(n_views: int, rank: int, world: int) -> List[int]:
    """Views of this rank: round-robin (v = rank, rank + world, ...).  Cameras of an orbit that are
    adjacent in index see similar instance counts, so round-robin balances the load better than blocks.
    Every view belongs to exactly one rank; a rank may get an empty list when world > n_views."""
    if n_views < 0 or world <= 0 or not (0 <= rank < world):
        raise ValueError(f"shard_views: bad arguments n_views={n_views} rank={rank} world={world}")
    return list(range(rank, n_views, world))


def max_over_ranks(value: float, device=None) -> float:
    """MAX over ranks of a per-rank scalar (device-timed milliseconds); identity when not distributed."""
    rank, world = world_info()
    if world == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def allreduce_accumulators(num: torch.Tensor, den: torch.Tensor, group=None) -> None:
    """In-place all-reduce(sum) of the fusion accumulators over all ranks: after it every rank holds the
    accumulators of ALL views and can finalise (f_i = num_i / den_i).  NCCL over NVLink/NVSwitch on GPUs.
    Must be called on the stream the accumulating fhgs_fuse_features calls were enqueued on (torch's
    current stream: NCCL orders itself after it)."""
    rank, world = world_info()
    if world == 1:
        return
    if num.dim() != 2 or den.dim() != 1 or num.shape[0] != den.shape[0]:
        raise ValueError("allreduce_accumulators: num must be [N,D] and den [N]")
    if not (num.is_contiguous() and den.is_contiguous()):
        raise ValueError("allreduce_accumulators: accumulators must be contiguous")
    dist.all_reduce(num, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(den, op=dist.ReduceOp.SUM, group=group)


def fuse_views_sharded(views: Sequence[int], fuse_one_view: Callable[[int, bool], None], num: torch.Tensor,
                       den: torch.Tensor, finalize: Callable[[], None],
                       before_reduce: Callable[[], None] | None = None) -> List[int]:
    """Driver of the view-sharded fusion.  `views` = all view indices; this rank handles shard_views of
    them.  `fuse_one_view(v, first)` must project + bin_sort view v and call fhgs_fuse_features to
    accumulate into (num, den), with FHGS_FUSE_ZERO when `first`; a rank with no view zeroes its
    accumulators itself.  Then one all-reduce, then `finalize()` (FHGS_FUSE_FINALIZE_ONLY) on every
    rank.  `before_reduce()` (optional) runs right before the all-reduce is enqueued (bench.py records a CUDA event
    there).  Returns the views this rank fused."""
    rank, world = world_info()
    mine = [views[i] for i in shard_views(len(views), rank, world)]
    if not mine:
        num.zero_()
        den.zero_()
    for k, v in enumerate(mine):
        fuse_one_view(v, k == 0)
    if before_reduce is not None:
        before_reduce()
    allreduce_accumulators(num, den)
    finalize()
    return mine
