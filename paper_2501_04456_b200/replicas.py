"""Multi-GPU = independent replicas.

The step does not shard without a per-step halo exchange that would cost as
much as the step itself at these sizes, and the paper's use is many
independent scenarios / seeds for hypothesis testing.  So
rank r runs its own replica of the workload with seed base+r on its own GPU;
there is NO data-path collective.  torch.distributed is used only for the
barrier and for the max-over-ranks / sum-over-ranks of the timing report.
The same functions run under gloo on CPU (tests/test_replicas.py).
"""
from __future__ import annotations

import os
from typing import Tuple


def env_rank_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of the replica on `rank`: distinct initial state AND noise key."""
    return int(base_seed) + 1000003 * int(rank)


def init(backend: str) -> None:
    import torch.distributed as dist
    if not dist.is_initialized():
        dist.init_process_group(backend=backend)


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def reduce_timing(elapsed_ms: float, units: float, device="cpu") -> Tuple[float, float]:
    """-> (max over ranks of elapsed_ms, sum over ranks of units).  Whole-job
    throughput = total units / slowest rank's time."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(elapsed_ms), float(units)
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())
