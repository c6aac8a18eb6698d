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


def _check_cuda_extension() -> None:
    """ReplicaSet is a product path: it fails loudly without the CUDA library
    (no CPU fallback)."""
    from . import binding
    binding.load()


class ReplicaSet:
    """R independent replicas of one workload on ONE GPU, each an `lv_sim`
    handle on its own CUDA stream ("batched replicas of
    small droplets" -- a C1- or Table-1-sized droplet, fills a
    fraction of a B200, and the paper's use is many scenarios / seeds for
    hypothesis testing).  `step(n)` enqueues the n graph
    replays of every replica in slices, round robin, so that every stream
    always has work queued and the kernels of different replicas overlap on
    the SMs.  With `batched=True` (default) the set is an `lv_batch` instead:
    ONE CUDA graph holds `steps_per_launch` steps of every replica as parallel
    branches, so a step of all R droplets is one launch, not 5 R.  There is no
    coupling between replicas: replica r of the set is bit-identical to the same
    workload stepped alone
    (tests/test_gpu_parity.py::test_replica_set_equals_solo_runs)."""

    def __init__(self, make_workload, n_replicas: int, base_seed: int, device: str = "cuda:0",
                 cells_per_cut=None, options=None, neighbour_list=None, slice_steps: int = 50,
                 batched: bool = True, steps_per_launch: int = 8):
        _check_cuda_extension()
        from . import binding, tuning
        if n_replicas < 1:
            raise ValueError("n_replicas must be >= 1")
        self.slice_steps = int(slice_steps)
        self.workloads = [make_workload(replica_seed(base_seed, r)) for r in range(n_replicas)]
        self.sims = [binding.Simulation.from_workload(
            w, cells_per_cut=cells_per_cut if cells_per_cut is not None else tuning.cells_per_cut(w),
            device=device, options=options, neighbour_list=neighbour_list) for w in self.workloads]
        self.batch = binding.Batch(self.sims, steps_per_launch) if batched else None

    def __len__(self) -> int:
        return len(self.sims)

    @property
    def n_particles(self) -> int:
        return sum(w.n for w in self.workloads)

    def step(self, n: int = 1) -> None:
        if self.batch is not None:
            self.batch.step(n)
            return
        done = 0
        while done < n:
            k = min(self.slice_steps, n - done)
            for s in self.sims:
                s.step(k)
            done += k

    def synchronize(self) -> None:
        for s in self.sims:
            s.synchronize()

    def get_state(self, r: int, **kw):
        return self.sims[r].get_state(**kw)

    def close(self) -> None:
        if getattr(self, "batch", None) is not None:
            self.batch.close()
            self.batch = None
        for s in self.sims:
            s.close()
        self.sims = []
