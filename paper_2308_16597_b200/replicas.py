"""Rank plumbing of the multi-GPU modes (replicas for the headline, y-slabs).

The path does not shard in this build (north_star: no sharding or collectives across GPUs):
under torchrun every rank runs an independent replica of the workload on its own GPU.  The only
cross-rank operations are the barrier around the timed region and the MAX of the device-measured
time, through `torch.distributed` (NCCL on the GPU box, gloo in the CPU tests).  Nothing of the
method's arithmetic lives here.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def rank_info():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str, device=None):
    """Joins the job's process group when WORLD_SIZE > 1 (rendezvous on 127.0.0.1 unless the
    launcher says otherwise); a no-op for a single process.  Returns world_size."""
    _, world, _ = rank_info()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=device)
        else:
            dist.init_process_group(backend)
    return world


def barrier(device=None):
    if dist.is_initialized():
        dist.barrier()
    if device is not None and torch.device(device).type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(value: float, device="cpu") -> float:
    """The slowest rank's value (every rank gets it)."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_mlups(nodes_per_replica: int, steps: int, ms_max: float, world: int) -> float:
    """Eq. (18) for the whole job: every replica's lattice updates over the
    slowest rank's time ("weak" scaling: per-GPU work is fixed)."""
    return world * nodes_per_replica * steps / (ms_max * 1e-3) / 1e6


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()
