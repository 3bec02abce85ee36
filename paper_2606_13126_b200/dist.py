"""Replica plumbing for bench.py --gpus N.  The path does not shard ("replicas only"): every rank
runs an independent replica of the workload (own seed) and there is NO data-path collective.  The only
communication is the timing protocol: a barrier on both sides of the timed region, MAX over ranks of the
device time, SUM over ranks of the processed units."""
from __future__ import annotations

import os

import torch
import torch.distributed as td


def env_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init(backend: str | None = None) -> tuple[int, int, int]:
    rank, local_rank, world = env_world()
    if world > 1 and not td.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29517")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
        td.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def _dev():
    return torch.device("cuda", torch.cuda.current_device()) if td.is_initialized() and td.get_backend() == "nccl" else torch.device("cpu")


def barrier() -> None:
    if td.is_initialized():
        td.barrier()


def max_over_ranks(x: float) -> float:
    if not td.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=_dev())
    td.all_reduce(t, op=td.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float) -> float:
    if not td.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=_dev())
    td.all_reduce(t, op=td.ReduceOp.SUM)
    return float(t.item())


def aggregate(units_this_rank: float, seconds_this_rank: float) -> dict:
    """Whole-job throughput: units all ranks processed / max-over-ranks time."""
    t = max_over_ranks(seconds_this_rank)
    u = sum_over_ranks(units_this_rank)
    return {"units": u, "seconds": t, "throughput": u / t if t > 0 else 0.0}


def shutdown() -> None:
    if td.is_initialized():
        td.destroy_process_group()
