"""View sharding for N > 1 GPUs: every view's preprocess -> sort -> forward -> backward is independent,
so rank r owns views r, r + world, ...; surfel parameters are replicated.  The only exchange step of the method is the
merge of the per-surfel visibility statistics at the end of a pruning interval ("rendering all
training views"): one all-reduce (sum) of vis_count / contrib_sum, after which every rank computes the same prune mask.
"""
from __future__ import annotations

from typing import List


def views_for_rank(n_views: int, rank: int, world: int) -> List[int]:
    if world <= 0 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    return list(range(rank, n_views, world))


def allreduce_stats(vis_count, contrib_sum):
    """In-place sum over ranks (NCCL for CUDA tensors, gloo for CPU tensors); no-op without a process group."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(vis_count, op=dist.ReduceOp.SUM)
        dist.all_reduce(contrib_sum, op=dist.ReduceOp.SUM)
    return vis_count, contrib_sum
