"""Multi-GPU plumbing: replicas only.

The path does not shard in this build: `bench.py --gpus N` runs N independent replicas, one process
per GPU, with no collective on the data path.  What the ranks share is the timing protocol: a
barrier on both sides of the timed region, the MAX over ranks of the device time, and the whole-job
throughput = units of all ranks / that time.  The functions take the process group explicitly so
that the same code runs over NCCL on GPUs and over gloo in the CPU tests (tests/test_replicas.py).
"""
from __future__ import annotations


def init(backend: str, rank: int, world: int, device=None):
    """torch.distributed process group for `world` replicas, or None when world == 1."""
    if world <= 1:
        return None
    import os
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29500")
    kwargs = {"device_id": device} if (device is not None and backend == "nccl") else {}
    dist.init_process_group(backend, rank=rank, world_size=world, **kwargs)
    return dist


def barrier(dist) -> None:
    if dist is not None:
        dist.barrier()


def max_over_ranks(value: float, dist, device="cpu") -> float:
    """MAX over the ranks of a per-rank scalar (the slowest replica defines the job time)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_mlups(cells: int, steps: int, world: int, ms: float) -> float:
    """lattice updates of ALL replicas per second / 1e6, for `ms` = max-over-ranks time of `steps` steps."""
    return world * cells * steps / (ms * 1e-3) / 1e6


def finish(dist) -> None:
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
