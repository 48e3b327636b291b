"""Host-side sharding logic for more than one GPU.

Reactors are independent, so a multi-GPU run is one process per GPU, each
evaluating its own reactors with no data-path collective.  The only communication is the timing
reduction: a multi-rank number is the MAX of the per-rank device times.  This module holds that
logic so that it can be tested on CPU with the gloo backend (tests/test_shard.py); bench.py uses it
with NCCL.  It contains none of the method's arithmetic.
"""
from __future__ import annotations


def state_seed(config_index: int, rank: int) -> int:
    """Seed of rank `rank`'s reactor states for config C<config_index> (weak scaling: every rank
    owns a full batch of its own; rank 0 is the single-GPU workload, seed 2000 + c)."""
    return 2000 + int(config_index) + 100 * int(rank)


def reactor_range(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous reactor range [lo, hi) of `rank` when ONE batch of n_total reactors is split over
    `world` ranks (strong scaling); sizes differ by at most one, lower ranks take the extra."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad rank/world/n_total")
    base, extra = divmod(int(n_total), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def max_over_ranks(value: float, device=None) -> float:
    """MAX over the ranks of the default process group (identity without one)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: int, steps: int, max_ms: float, world: int) -> float:
    """Units per second of the whole job: every rank processed units_per_rank units per step, the job
    took max_ms (the slowest rank) for `steps` steps."""
    return world * units_per_rank * steps / (max_ms * 1e-3)
