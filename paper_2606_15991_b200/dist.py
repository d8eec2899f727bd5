"""One-process-per-GPU plumbing for bench.py: rendezvous from the torchrun environment,
barrier, and max / sum over ranks.  The hot path has no exchange step (every output tile is an
independent unit), so N > 1 means N independent problems -- weak scaling --
and no data-path collective exists; torch.distributed carries only timing scalars."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(
        os.environ.get("WORLD_SIZE", "1"))


def init(backend: str | None = None):
    rank, local_rank, world_size = world()
    if world_size > 1 and not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        kwargs = {}
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
            kwargs["device_id"] = torch.device("cuda", local_rank)
        dist.init_process_group(backend=backend, rank=rank, world_size=world_size, **kwargs)
    return rank, local_rank, world_size


def _scalar_device():
    if dist.is_initialized() and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def barrier():
    if dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float) -> float:
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_scalar_device())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float) -> float:
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_scalar_device())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def units_for_rank(n_units: int, rank: int, world_size: int):
    """Contiguous, balanced share of `n_units` independent units (strong-scaling helper)."""
    base, rem = divmod(n_units, world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()
