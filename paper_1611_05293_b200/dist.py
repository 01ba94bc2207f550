"""Multi-GPU plumbing: one process per GPU, `torch.distributed` for rendezvous, barrier and the
max-over-ranks of the timed region.  The split step of ONE simulation does not shard (every step
needs the whole profile and a replicated wake); independent simulations
(a batched scan, or replicas) are partitioned across ranks with NO data-path collective.
"""
from __future__ import annotations

import os
from typing import List, Sequence, Tuple


def env_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str) -> Tuple[int, int, int]:
    """Join the process group named by MASTER_ADDR/MASTER_PORT (no-op for a single process)."""
    rank, local_rank, world = env_world()
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29500")
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def shutdown() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def reduce_max(value: float, device=None) -> float:
    """max over ranks of a host scalar (the timed region of a multi-GPU run)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_sum(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def shard_members(members: int, rank: int, world: int) -> List[int]:
    """Contiguous, balanced partition of batch members 0..members-1; the first (members % world)
    ranks get one more.  Ranks beyond `members` get an empty list."""
    if members < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad shard request")
    base, extra = divmod(members, world)
    lo = rank * base + min(rank, extra)
    return list(range(lo, lo + base + (1 if rank < extra else 0)))


def replica_seeds(seeds: Sequence[int], rank: int) -> Tuple[int, ...]:
    """Replica mode: rank r runs the same workload with its seeds shifted by 7919*r, so the
    replicas are independent simulations rather than copies."""
    return tuple(int(s) + 7919 * rank for s in seeds)
