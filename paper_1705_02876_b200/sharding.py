"""Multi-GPU plumbing: the path shards by event with no data-path collective.

Tracks and candidates are independent, and hit bins are per event and layer, so rank r simply owns a
contiguous range of events.  torch.distributed is used only for the rendezvous, the barrier around the
timed region and the max-over-ranks reduction of the measured time (NCCL on GPUs, gloo in CPU tests).
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def world() -> tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str | None = None) -> tuple[int, int, int]:
    rank, local_rank, ws = world()
    if ws > 1 and not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        kw = {}
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
            kw["device_id"] = torch.device("cuda", local_rank)
        dist.init_process_group(backend=backend, rank=rank, world_size=ws, **kw)
    return rank, local_rank, ws


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()


def events_of_rank(events_per_rank: int, rank: int) -> range:
    """Weak scaling: every rank fits its own `events_per_rank` events (global event ids)."""
    return range(rank * events_per_rank, (rank + 1) * events_per_rank)


def split_events(n_events: int, rank: int, world_size: int) -> range:
    """Strong scaling: a fixed set of events cut into contiguous, near-equal ranges."""
    lo = n_events * rank // world_size
    hi = n_events * (rank + 1) // world_size
    return range(lo, hi)


def barrier(device=None):
    if dist.is_initialized():
        if device is not None and torch.device(device).type == "cuda":
            dist.barrier(device_ids=[torch.device(device).index])
        else:
            dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
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
