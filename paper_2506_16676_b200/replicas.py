"""Multi-GPU plumbing of ``bench.py``: REPLICAS ONLY.

The solve path does not shard (BASELINE.json north_star: "one GPU only: no sharding, no inter-GPU
collectives").  ``bench.py --gpus N`` therefore runs N independent replicas of the
same solve, one process per GPU, and the only communication is the timing protocol of the bench contract:
a barrier on both sides of the timed region and the MAX over ranks of the device time.  Works with the
``nccl`` backend on GPUs and with ``gloo`` on CPU (tests/test_replicas.py, world_size 2).
"""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process: 0, 0, 1)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str):
    """Initialise torch.distributed from the env if WORLD_SIZE > 1.  Returns (rank, local_rank, world_size)."""
    rank, local_rank, world = env_world()
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX over ranks of a per-rank scalar (the bench contract's timing rule); identity for one process."""
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


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
