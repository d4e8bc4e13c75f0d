"""Multi-GPU plumbing of the benchmark: REPLICAS ONLY.

Configurations are independent and the tables are a few KiB, so the path has no exchange step and
`north_star` restricts the build to one GPU per job: with N ranks every rank integrates the whole
workload on its own GPU.  The only communication is the timing protocol of bench.py: a barrier on
both sides of the timed region and the MAX over ranks of the device time.  These helpers hold that
protocol so that it can be tested on CPU with the gloo backend (tests/test_replicas_gloo.py).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world_size() -> int:
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def rank() -> int:
    return dist.get_rank() if dist.is_available() and dist.is_initialized() else 0


def barrier() -> None:
    if world_size() > 1:
        dist.barrier()


def max_over_ranks(seconds: float, device: torch.device | str = "cpu") -> float:
    """MAX over ranks of a locally measured duration (the slowest replica defines the step time)."""
    if world_size() == 1:
        return float(seconds)
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_runs(workload):
    """Runs a rank executes: all of them (replicas); kept as a function so the plan is explicit."""
    return list(workload.runs)


def whole_job_rate(units_per_replica_step: int, steps: int, seconds_max: float) -> float:
    """Aggregate rate over all replicas: every rank did `units_per_replica_step * steps` units in the
    time of the slowest one."""
    return world_size() * units_per_replica_step * steps / seconds_max
