"""Multi-GPU plumbing for the replica (weak-scaling) layout: one process per GPU, each rank runs the split MLP
on its own token batch; no data-path collective.  torch.distributed is used only to line ranks up
and to take the max over ranks of the device time.  Works with NCCL (GPU) and gloo (CPU tests)."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_world():
    """(world_size, rank, local_rank) from the torchrun environment; (1, 0, 0) when not launched by it."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def rank_seed(base_seed: int, rank: int) -> int:
    """Rank r draws its own token batch and (replicated-shape) weights from seed base + r."""
    return base_seed + rank


def init(backend: str | None = None):
    world, rank, local = env_world()
    if world > 1 and not dist.is_initialized():
        backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
        if backend == "nccl":
            torch.cuda.set_device(local)
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
    elif torch.cuda.is_available():
        torch.cuda.set_device(local if world > 1 else 0)
    return world, rank, local


def _device():
    return torch.device("cuda") if (dist.is_initialized() and dist.get_backend() == "nccl") else torch.device("cpu")


def barrier():
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
    if torch.cuda.is_available():
        torch.cuda.synchronize()


def max_over_ranks(x: float) -> float:
    if dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([x], dtype=torch.float64, device=_device())
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())
    return float(x)


def whole_job_throughput(local_ms_per_step: float, units_per_rank_per_step: float) -> tuple[float, float]:
    """(units/s summed over all ranks, max-over-ranks ms per step): every rank processes the same number of
    units per step, the job's step time is the slowest rank's."""
    world = dist.get_world_size() if dist.is_initialized() else 1
    ms = max_over_ranks(local_ms_per_step)
    return world * units_per_rank_per_step / (ms * 1e-3), ms


def finalize():
    if dist.is_initialized():
        dist.destroy_process_group()
