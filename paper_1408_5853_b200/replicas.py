"""Multi-GPU host logic: replicas only.

BASELINE.json fixes the build to one GPU, and the path has no exchange step that is built, so
`bench.py --gpus N` runs N independent replicas of the workload, one process per GPU, with no
data-path collective.  The only communication is the measurement protocol: a barrier on both
sides of the timed region and the MAX over ranks of the device-timed duration.  This module holds
that protocol so that it can be tested with the gloo backend on CPU (tests/test_replicas.py).
"""
from __future__ import annotations

import os


def rank_env():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) without it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str, local_rank: int, world: int):
    """torch.distributed process group for world > 1 (nccl on GPUs, gloo in the CPU tests); None for 1."""
    if world <= 1:
        return None
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        kw = {"device_id": torch.device("cuda", local_rank)} if backend == "nccl" else {}
        dist.init_process_group(backend, **kw)
    return dist


def barrier(dist, sync=None):
    """Barrier over the ranks, then the local device synchronize (`sync`, e.g. torch.cuda.synchronize)."""
    if dist is not None:
        dist.barrier()
    if sync is not None:
        sync()


def max_over_ranks(x: float, dist, device="cpu") -> float:
    """MAX over ranks of a locally measured duration (every rank gets the result)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_gcups(cells_per_replica: int, steps: int, seconds_max: float, world: int) -> float:
    """Whole-job throughput of `world` replicas that each advanced `cells_per_replica` cells by
    `steps` steps within `seconds_max` (the slowest rank's time): weak scaling."""
    return world * cells_per_replica * steps / seconds_max / 1e9
