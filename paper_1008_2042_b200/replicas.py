"""Multi-GPU plumbing for the "replicas only" mode: the hot path does not shard
(north_star: one GPU, no collectives), so N GPUs run N independent reconstructions.  The only
cross-rank traffic is the timing protocol of bench.py: a barrier on both sides of the timed region
and the MAX over ranks of the device time.  Backend nccl on GPUs, gloo in the CPU tests."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def world():
    """(rank, world_size, local_rank) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str = "nccl", device=None) -> None:
    rank, size, _ = world()
    if size > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        kw = {}
        if backend == "nccl" and device is not None:
            kw["device_id"] = device
        dist.init_process_group(backend, rank=rank, world_size=size, **kw)


def barrier(device=None) -> None:
    if dist.is_initialized():
        dist.barrier()
    if device is not None and torch.device(device).type == "cuda":
        torch.cuda.synchronize()


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX over ranks of a per-rank scalar (the job takes as long as its slowest replica)."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_replica: float, seconds_local: float, device="cpu") -> float:
    """Whole-job throughput of N identical replicas: N * units / max_r(seconds_r)."""
    n = dist.get_world_size() if dist.is_initialized() else 1
    return n * units_per_replica / max_over_ranks(seconds_local, device)


def shutdown() -> None:
    if dist.is_initialized():
        dist.destroy_process_group()
