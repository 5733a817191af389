"""Host-side plumbing for N > 1: independent replicas, one process per GPU (DESIGN.md s4 'replicas only').

The path of BASELINE.json is scoped to one GPU (K partitions = K simulated ranks on that GPU), so N
GPUs run N independent replicas of the whole iteration on different seeded views: no data-path
collective exists.  What remains for `torch.distributed` is the measurement protocol of bench.py:
a barrier on both sides of the timed region, the MAX over ranks of the device time, and the
whole-job throughput = units all ranks processed / that time.  Backend `nccl` on GPUs, `gloo` in
the CPU tests (tests/test_replicas.py, world_size 2).
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def world_info():
    """(world_size, rank, local_rank) from the torchrun environment (1, 0, 0 when absent)."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str, local_rank: int = 0):
    """Join the job if there is more than one rank; returns (world, rank)."""
    world, rank, _ = world_info()
    if world > 1 and not dist.is_initialized():
        kw = {}
        if backend == "nccl":
            kw["device_id"] = torch.device("cuda", local_rank)
        dist.init_process_group(backend, **kw)
    return world, rank


def finish():
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()


def barrier(cuda: bool):
    """Device-quiet on both sides of a rendezvous (the bench contract's bracket)."""
    if cuda:
        torch.cuda.synchronize()
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
    if cuda:
        torch.cuda.synchronize()


def max_over_ranks(value: float, cuda: bool) -> float:
    """MAX over ranks of a per-rank time (ms)."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device="cuda" if cuda else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, cuda: bool) -> float:
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device="cuda" if cuda else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def replica_view_seed(base_seed: int, rank: int) -> int:
    """Every replica trains on its own seeded view (weak scaling: per-GPU work fixed)."""
    return int(base_seed) + 7919 * int(rank)


def shard_views(n_views: int, world: int, rank: int):
    """Round-robin assignment of the views of a batch to replicas (used when B views are spread over GPUs)."""
    return list(range(rank, n_views, world))


def whole_job_throughput(units_this_rank: float, ms_this_rank: float, cuda: bool):
    """(units of all ranks / max-over-ranks time in s, max-over-ranks ms)."""
    ms = max_over_ranks(ms_this_rank, cuda)
    units = sum_over_ranks(units_this_rank, cuda)
    return units / (ms * 1e-3), ms
