"""Multi-GPU plumbing: the path shards over parameter vectors with no exchange.

Every (parameter vector, exposure) is independent, so each rank owns a slice
of the pv axis - rows of ``pv``, ``ldp``, the table and ``flux`` - and replicates the small shared
inputs (geometry weights, times, light-curve tags).  No collective sits on the data path; the only
communication is the barrier and the max-over-ranks of the device time that ``bench.py`` reports.
Host logic only (no model arithmetic): covered by world_size-2 gloo tests on CPU.
"""
from __future__ import annotations

import os


def pv_slice(npv: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [begin, end) of the pv axis owned by ``rank``; sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world) or npv < 0:
        raise ValueError("bad rank/world/npv")
    base, extra = divmod(npv, world)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def env_rank() -> tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init_process_group(backend: str):
    """Join the job's process group if launched under torchrun with more than one rank."""
    import torch.distributed as dist
    rank, _, world = env_rank()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (the device time of the timed region)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """Sum of a per-rank scalar (units processed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
