"""Replica plumbing for N > 1 ("replicas only").

north_star forbids sharding and halo exchange (BASELINE.json:5), so the N-GPU job is N independent copies of the
same single-GPU path — one process per GPU, no data-path collective.  The only things that cross ranks are the
barrier around the timed region and the MAX of the per-rank device times; this module holds exactly that, so that
`bench.py` (NCCL, one GPU per rank) and the CPU tests (gloo, world_size 2) run the same code.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env():
    """(rank, local_rank, world) from the torchrun environment; (0, 0, 1) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str | None = None, device: torch.device | None = None) -> int:
    """Join the process group when WORLD_SIZE > 1 (MASTER_ADDR / MASTER_PORT from the environment).  Returns world."""
    _, _, world = env()
    if world > 1 and not dist.is_initialized():
        backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
        kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
        dist.init_process_group(backend, **kw)
    return world


def _device() -> torch.device:
    if dist.is_initialized() and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def barrier() -> None:
    """Process-group barrier (if any) followed by a device synchronise (if a device is in use)."""
    if dist.is_initialized():
        dist.barrier()
    if torch.cuda.is_available():
        torch.cuda.synchronize()


def max_over_ranks(value: float) -> float:
    """MAX of a per-rank scalar (a device time): the job is as slow as its slowest replica."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, seconds_this_rank: float) -> float:
    """Weak-scaling aggregate: every rank processed `units_per_rank`; rate = world * units / max-over-ranks time."""
    world = dist.get_world_size() if dist.is_initialized() else 1
    return world * units_per_rank / max_over_ranks(seconds_this_rank)


def finish() -> None:
    if dist.is_initialized():
        dist.barrier()
        dist.destroy_process_group()
