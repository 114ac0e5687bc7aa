"""Multi-GPU plumbing: voices are independent and a sound is a pure function of
(seed, global voice index), so the path shards by batch index with NO data-path collective.  One process
per GPU; torch.distributed is used only for the barrier and the max-over-ranks timing."""
from __future__ import annotations

import os


def world():
    """(rank, local_rank, world_size) from the torchrun environment (1-process defaults)."""
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def batch_index(step: int, rank: int, world_size: int, first: int = 0) -> int:
    """Weak scaling: at every step each rank renders its own batch; indices are disjoint and dense."""
    return first + step * world_size + rank


def init(backend: str):
    import torch.distributed as dist
    rank, local_rank, ws = world()
    if backend == "nccl":          # one process per GPU: bind the device before NCCL picks one
        import torch
        torch.cuda.set_device(local_rank)
    if ws > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=ws)
    return rank, local_rank, ws


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
