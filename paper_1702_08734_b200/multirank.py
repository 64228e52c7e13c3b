"""Host logic of the N > 1 runs (one process per GPU, torch.distributed).

The hot path partitions by rows / queries (replicas, "near linear speedup"), so
there is no data-path collective: every rank runs the same calls on its own rows.  The
only communication is the barrier around the timed region and the max-over-ranks of the
device time; the job's value is the sum of the ranks' work divided by that time.
Backend-agnostic (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def rank_rows(rank: int, rows_per_rank: int) -> tuple[int, int]:
    """(first global row, number of rows) of a rank: weak scaling, disjoint consecutive ranges."""
    return rank * rows_per_rank, rows_per_rank


def world() -> tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def barrier() -> None:
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def max_over_ranks(x: float, device="cpu") -> float:
    """The slowest rank's time: what a job that waits for all ranks observes."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: float, ms_per_step_max: float, world_size: int) -> float:
    """Whole-job units per second: all ranks' units over the slowest rank's step time."""
    return world_size * units_per_rank / (ms_per_step_max * 1e-3)
