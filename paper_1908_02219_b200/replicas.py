"""Multi-GPU = independent replicas: BASELINE.json's north_star scopes
the deposition to one GPU with no sharding and no collective, so `bench.py --gpus N` runs N
independent copies of the single-GPU path, one process per GPU, each on its own seeded marker
set.  The only cross-rank traffic is this bookkeeping: a barrier around the timed region, the
MAX of the per-rank device times and the SUM of the per-rank units.  No data-path collective.

Works with any torch.distributed backend (nccl on the GPU box; gloo in the CPU tests).
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) if absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str | None = None):
    """Initialises torch.distributed when WORLD_SIZE > 1.  Returns (rank, local_rank, world)."""
    rank, local_rank, world = env_rank()
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            kw = {}
            if backend == "nccl":
                torch.cuda.set_device(local_rank)
                kw["device_id"] = torch.device("cuda", local_rank)
            dist.init_process_group(backend=backend, rank=rank, world_size=world, **kw)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def combine(elapsed_ms: float, units: float, device="cpu"):
    """Whole-job figures over all replicas: (max over ranks of elapsed_ms, sum over ranks of
    units).  Identity when not distributed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(elapsed_ms), float(units)
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def replica_seed(base_seed: int, rank: int) -> int:
    """Each replica deposits its own markers (same distributions, different seed)."""
    return base_seed + 1_000_003 * rank


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
