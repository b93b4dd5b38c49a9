"""View sharding for N > 1 GPUs: every view's preprocess -> sort -> forward -> backward is independent,
so rank r owns views r, r + world, ...; surfel parameters are replicated and the per-view step needs no collective.
The method has two real exchange steps, both plain sums over ranks (NCCL over NVLink for CUDA tensors, gloo on CPU):
  * the merge of the per-surfel visibility statistics at the end of a pruning interval (PAPER.md:219
    "rendering all training views"): one all-reduce of vis_count / contrib_sum, after which every rank computes the same
    prune mask (the compaction is deterministic, so the replicas stay in lock-step);
  * when `world` views are batched into one optimiser step (a change of optimisation semantics against the paper's one view
    per iteration): one all-reduce of the 58 N gradient floats per step.
This module holds that bookkeeping (no arithmetic of the method) and the launcher bench.py uses for `--gpus N`.
"""
from __future__ import annotations

import os
import subprocess
import sys
from typing import Dict, List, Optional


def views_for_rank(n_views: int, rank: int, world: int) -> List[int]:
    if world <= 0 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    return list(range(rank, n_views, world))


def rotation_for_rank(n_views: int, rank: int, world: int, per_rank: int) -> List[int]:
    """The views rank `rank` rotates over in a benchmark or an epoch: its shard r, r + world, ..., cut to `per_rank` views
    (0 = the whole shard).  Never empty: with more ranks than views the extra ranks repeat views (rank mod n_views)."""
    mine = views_for_rank(n_views, rank, world)
    if per_rank > 0:
        mine = mine[:per_rank]
    return mine or [rank % n_views]


def _group_active() -> bool:
    import torch.distributed as dist
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def allreduce_stats(vis_count, contrib_sum):
    """In-place sum over ranks (NCCL for CUDA tensors, gloo for CPU tensors); no-op without a process group."""
    import torch.distributed as dist
    if _group_active():
        dist.all_reduce(vis_count, op=dist.ReduceOp.SUM)
        dist.all_reduce(contrib_sum, op=dist.ReduceOp.SUM)
    return vis_count, contrib_sum


def allreduce_grads(grads: Dict[str, "object"]):
    """Batched-view mode: in-place sum over ranks of every gradient array of the step (d_pos, d_scale, d_quat, d_opacity,
    d_sh; d_center2d too when present -- its norm is accumulated per view, so it is summed like the rest); no-op without
    a process group.  Returns the number of bytes reduced per rank."""
    import torch.distributed as dist
    nbytes = 0
    for k in sorted(grads):
        t = grads[k]
        nbytes += t.numel() * t.element_size()
        if _group_active():
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return nbytes


def max_over_ranks(value: float, device=None) -> float:
    """Timing rule of the bench: a multi-GPU number is the MAX over ranks of the device-measured time."""
    import torch
    import torch.distributed as dist
    if not _group_active():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank_step: float, world: int, ms_per_step_max: float) -> float:
    """Whole-job units per second: every rank processes `units_per_rank_step` per step, all ranks step concurrently."""
    return units_per_rank_step * world / (ms_per_step_max * 1e-3)


def env_rank() -> tuple:
    """(rank, world, local_rank) from the torchrun environment; (0, 1, 0) when not launched by it."""
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def relaunch_under_torchrun(n_gpus: int, argv: List[str], available: Optional[int] = None) -> Optional[int]:
    """`python bench.py --gpus N` with N > 1 outside torchrun: start N ranks of this same command on this node
    (`python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 ...`) and return the exit code.
    Returns None when nothing is to be done (N == 1, or already inside a torchrun launch).  Raises RuntimeError when the
    node has fewer than N CUDA devices: a multi-GPU number is never measured on fewer GPUs than it names."""
    if n_gpus <= 1 or "WORLD_SIZE" in os.environ:
        return None
    if available is None:
        import torch
        available = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if available < n_gpus:
        raise RuntimeError(f"--gpus {n_gpus} needs {n_gpus} CUDA devices on this node, found {available}")
    port = 29500 + (os.getpid() % 2000)
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")  # the communicator lines (rings / trees / NVLS) stay visible on stderr
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port)] + argv
    return subprocess.call(cmd, env=env)
