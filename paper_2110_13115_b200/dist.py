"""Multi-GPU plumbing for bench.py: one process per GPU, no data-path collective.

The hot path has no exchange step ("several" GPUs each filter their own data segments with
the basis and coefficients resident; throughput is quoted per GPU).  So N ranks = N independent strain segments
against the same bank ("weak" scaling); torch.distributed is used only for the barrier and the max-over-ranks of the
device-measured time.  Backend nccl on GPUs, gloo in the CPU tests.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when not launched by torchrun."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str | None = None) -> tuple[int, int, int]:
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def segment_index(rank: int, step: int, world: int) -> int:
    """Which strain segment rank `rank` filters at step `step`: segments are dealt round-robin, so the job as a
    whole filters world * steps distinct consecutive segments."""
    return step * world + rank


def barrier(device=None):
    if dist.is_initialized():
        if device is not None and torch.device(device).type == "cuda":
            dist.barrier(device_ids=[torch.device(device).index])
        else:
            dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (the device-measured elapsed time)."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def finalize():
    if dist.is_initialized():
        dist.destroy_process_group()
