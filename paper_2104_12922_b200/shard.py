"""Multi-GPU plumbing: voices are independent and a sound is a pure function of
(seed, global voice index), so the path shards by batch index with NO data-path collective.  One process
per GPU; torch.distributed is used only for the barrier and the max-over-ranks timing.

Partition ("contiguous ranges of batch_index per GPU"): rank r owns the batch indices
[first + r*per_rank, first + (r+1)*per_rank); its step s renders index first + r*per_rank + s."""
from __future__ import annotations

import os
import socket
import subprocess
import sys


def world():
    """(rank, local_rank, world_size) from the torchrun environment (1-process defaults)."""
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def under_torchrun() -> bool:
    return "RANK" in os.environ and "WORLD_SIZE" in os.environ


def batch_range(rank: int, world_size: int, per_rank: int, first: int = 0):
    """-> (first batch index, count) of this rank's contiguous range."""
    if not (0 <= rank < world_size) or per_rank < 0:
        raise ValueError("bad rank / per_rank")
    return first + rank * per_rank, per_rank


def batch_index(step: int, rank: int, world_size: int, per_rank: int, first: int = 0) -> int:
    """Batch index of this rank's step `step` (0 <= step < per_rank): ranges are disjoint and dense over the ranks."""
    start, count = batch_range(rank, world_size, per_rank, first)
    if not (0 <= step < count):
        raise ValueError("step outside this rank's range")
    return start + step


def free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def launch_cmd(n: int, script: str, args, port: int):
    """The torchrun command line that starts `script args` as n ranks on this node (rendezvous on 127.0.0.1)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
            "--master-port", str(port), script] + list(args)


def respawn_under_torchrun(n: int, script: str, args, require_gpus: bool = True) -> int:
    """`python bench.py --gpus N` outside torchrun: start the N ranks ourselves.  Fails loudly if the node has fewer than
    N CUDA devices (never runs fewer ranks than asked for).  -> the launcher's exit code."""
    if n < 1:
        raise SystemExit("--gpus must be >= 1")
    if require_gpus:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < n:
            raise SystemExit(f"--gpus {n} asked for, but this node has {have} CUDA device(s)")
    env = dict(os.environ)
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    return subprocess.call(launch_cmd(n, script, args, free_port()), env=env)


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
