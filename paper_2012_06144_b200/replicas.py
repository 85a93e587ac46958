"""Multi-GPU plumbing for the "replicas only" mode.

The coupled ACM step does not shard in this build (north_star: one GPU, no collectives), so N ranks
run N independent replicas.  torch.distributed is used only for the barrier around the timed
region and for the max-over-ranks of the device time; there is no data-path collective.
Works with backend "nccl" (one rank per GPU, bench.py) and "gloo" (CPU tests).
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_ranks():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str, device=None):
    """Joins the process group described by RANK/WORLD_SIZE/MASTER_* if WORLD_SIZE > 1."""
    rank, local_rank, world = env_ranks()
    if world > 1 and not dist.is_initialized():
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=device)
        else:
            dist.init_process_group(backend)
    return rank, local_rank, world


def barrier(device=None):
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
    if device is not None and torch.device(device).type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(value: float, device=None) -> float:
    """Slowest rank's time: every multi-GPU number is reported as the max over ranks."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    on_host = device is None or dist.get_backend() != "nccl"      # gloo reduces host tensors
    t = torch.tensor([float(value)], dtype=torch.float64, device="cpu" if on_host else device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_mlups(cells_per_replica: int, steps: int, ms_max: float, world: int) -> float:
    """Whole-job throughput: lattice updates of all replicas / slowest rank's time (weak scaling)."""
    return world * cells_per_replica * steps / (ms_max * 1e-3) / 1e6


def shutdown():
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
