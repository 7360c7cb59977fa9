"""Multi-GPU = replicas only.

The N-turn sweeps alternate between turn curves (which span every Theta and wander +-R in x, y) and straight
lines (which span the full x or y extent of one Theta slice), so no partition of the volume survives two
consecutive kernels without a full re-shard; the independent unit is a whole plan.  One process per GPU,
one planner handle per process, no data-path collective.  The only communication is the bench contract's
barrier and the max-over-ranks / sum-over-ranks of two scalars, which this module provides for both the
`nccl` (GPU box) and `gloo` (CPU tests) backends.
"""
from __future__ import annotations

import os


def world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when launched plainly."""
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def init(backend: str):
    """Join the process group described by RANK / WORLD_SIZE / MASTER_ADDR / MASTER_PORT (no-op for one rank)."""
    rank, local_rank, ws = world()
    if ws > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            dist.init_process_group(backend=backend, rank=rank, world_size=ws)
    return rank, local_rank, ws


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def aggregate(ms_local: float, units_local: float, device="cpu"):
    """Whole-job figures of a replica run: (max over ranks of the elapsed ms, sum over ranks of the units)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(ms_local), float(units_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def replica_seed(config: int, rank: int) -> int:
    """Scene seed of a replica: rank 0 plans the named config (seed = config number), rank r > 0 plans another
    scene of the same class (same sizes and work, different obstacles / start / goal)."""
    return config + 1000 * rank


def shutdown():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
