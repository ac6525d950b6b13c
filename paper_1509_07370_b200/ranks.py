"""Multi-GPU plumbing of the benchmark: the path does not shard in this scope (DESIGN.md "Multi-GPU":
replicas only), so N ranks run N independent replicas and the only cross-rank step is the timing
reduction -- the slowest rank's device time decides, the whole job's rate counts every rank's cells.
No method arithmetic lives here."""
from __future__ import annotations


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX of a list of floats over all ranks (identity without a process group)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def whole_job_rate(units_per_rank: int, steps: int, seconds_max: float, world: int) -> float:
    """Units processed by ALL ranks per second of the slowest rank (weak scaling: every rank does
    `units_per_rank` units per step)."""
    return world * units_per_rank * steps / seconds_max
