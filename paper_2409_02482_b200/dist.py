"""Multi-GPU plumbing for the renderer: the path shards by camera batch with NO data-path collective
(DESIGN.md §9): every rank holds the whole scene and renders its own batch of views; the only
communication is the barrier and the max-over-ranks reduction of the timing.  torch.distributed
(nccl on GPUs, gloo in the CPU tests) is plumbing only."""
from __future__ import annotations

import math
import os


def env_rank():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init_process_group(backend: str):
    import torch.distributed as dist
    rank, _, world = env_rank()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def rank_camera_rotation(rank: int, world: int) -> float:
    """Weak scaling: every rank renders a batch of the SAME size; rank r's Fibonacci camera lattice
    is rotated about the vertical axis so that the ranks look at different views."""
    return 0.0 if world <= 1 else 2.0 * math.pi * rank / (world * 64.0)


def shard_views(num_views: int, rank: int, world: int):
    """Strong-scaling helper: contiguous, balanced split of one camera batch across ranks."""
    base, rem = divmod(num_views, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_throughput(units_this_rank: float, seconds_this_rank: float, device="cpu") -> float:
    """units all ranks processed / max-over-ranks time."""
    return sum_over_ranks(units_this_rank, device) / max_over_ranks(seconds_this_rank, device)
