"""Multi-GPU plumbing: jobs are independent units living in host memory, so the path shards by
job with NO data-path collective -- one scheduler instance per GPU, one process per GPU.  The only communication is
the timing reduction (max over ranks) and the unit count (sum over ranks), both over torch.distributed.
Works with the `nccl` backend on GPUs and with `gloo` on CPU (tests/test_multi_rank.py, world_size 2).
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when launched plainly."""
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def shard_jobs(num_jobs: int, rank: int, world: int, scaling: str = "weak"):
    """Global job ids rank `rank` owns.
    weak  : every rank runs `num_jobs` jobs of its own (ids rank*num_jobs ...), per-GPU work fixed as N grows.
    strong: the `num_jobs` jobs are dealt round-robin (home GPU = job_id mod world)."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError((rank, world))
    if scaling == "weak":
        return range(rank * num_jobs, (rank + 1) * num_jobs)
    if scaling == "strong":
        return range(rank, num_jobs, world)
    raise ValueError(scaling)


def init_process_group(backend: str | None = None):
    """Join the job's process group when WORLD_SIZE > 1 (MASTER_ADDR/PORT from the environment)."""
    import torch.distributed as dist
    rank, local_rank, world = env_rank()
    if world > 1 and not dist.is_initialized():
        if backend is None:
            import torch
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier(device=None):
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        if device is not None and str(device).startswith("cuda"):
            import torch
            dist.barrier(device_ids=[torch.device(device).index or 0])
        else:
            dist.barrier()


def aggregate(ms_local: float, units_local: float, device="cpu"):
    """(max over ranks of the step time in ms, sum over ranks of the units processed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(ms_local), float(units_local)
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())
