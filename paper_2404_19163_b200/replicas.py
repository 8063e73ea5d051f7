"""Multi-GPU = independent replicas: one refinement is a chain of dependent
dense GEMMs over the same operands and does not shard; N GPUs run N independent problems (the
graph-partitioned sub-problems of PAPER.md:98) with NO data-path collective.  This module only
holds the rendezvous and the timing aggregation (max over ranks) used by bench.py."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init(backend: str | None = None) -> tuple[int, int, int]:
    """Initialise torch.distributed from the torchrun environment (no-op for world size 1)."""
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier() -> None:
    if dist.is_initialized():
        dist.barrier()


def aggregate(elapsed_ms: float, units: float, device: str | torch.device = "cpu") -> tuple[float, float]:
    """(max over ranks of elapsed_ms, sum over ranks of units): whole-job throughput of N
    independent replicas is sum(units) / max(time)."""
    if not dist.is_initialized():
        return float(elapsed_ms), float(units)
    if dist.get_backend() == "gloo":
        device = "cpu"
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def shutdown() -> None:
    if dist.is_initialized():
        dist.destroy_process_group()
