"""Multi-GPU plumbing for the marker push.

Markers are independent, so the path shards by markers with NO data-path
collective: rank r owns a contiguous block of the global marker stream, mesh and coefficient
tables are replicated on every GPU.  The only communication is bookkeeping: the max over
ranks of the device-timed duration, and sums of counters.  Works with any torch.distributed
backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import Dict, Tuple

import torch
import torch.distributed as dist


def env_rank() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str = "nccl") -> Tuple[int, int, int]:
    rank, local_rank, world = env_rank()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def shard_range(n_global: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous block [lo, hi) of rank `rank`; blocks differ by at most one marker."""
    base, rem = divmod(int(n_global), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def rank_seed(seed: int, rank: int) -> int:
    """Weak scaling: every rank draws its own n markers from an independent stream."""
    return int(seed) + 1000003 * int(rank)


def barrier():
    if dist.is_initialized():
        dist.barrier()


def reduce_max(x: float, device="cpu") -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_sum(x: float, device="cpu") -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def allreduce_sum_(t: torch.Tensor) -> torch.Tensor:
    """In-place sum over ranks: the ONE data-path collective of the PIC cycle's particle side -- the right-hand side of
    trimeg_scatter (row f1: every GPU projects its own markers, the [n_modes][n_vert][6] complex vector is summed; <= 60 MB
    for the largest config).  complex tensors are reduced through their real view (NCCL has no complex type)."""
    if dist.is_initialized():
        dist.all_reduce(torch.view_as_real(t) if t.is_complex() else t, op=dist.ReduceOp.SUM)
    return t


def aggregate(units_local: float, seconds_local: float, counters: Dict[str, int], device="cpu") -> Dict[str, float]:
    """Whole-job numbers: units summed over ranks, time = max over ranks, counters summed."""
    out = dict(units=reduce_sum(units_local, device), seconds=reduce_max(seconds_local, device))
    for k, v in counters.items():
        out[k] = reduce_sum(float(v), device)
    out["value"] = out["units"] / out["seconds"] if out["seconds"] > 0 else 0.0
    return out
