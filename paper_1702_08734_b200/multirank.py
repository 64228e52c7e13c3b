"""Host logic of the N > 1 runs (one process per GPU, torch.distributed).

Two ways to use G GPUs:
  replicas  the hot path partitions by rows / queries ("near linear speedup"): every rank runs
            the same calls on its own rows, no data-path collective (rank_rows);
  shards    the database is cut into G contiguous id ranges, every rank answers the FULL query batch
            over its shard, the [nq][k] (distance, id) lists are exchanged with ONE all-gather and
            merged by "an additional round of k-selection": sharded_search / merge.
The barrier and the max-over-ranks of the device time bracket the timed region of bench.py.
Backend-agnostic (nccl on GPUs, gloo in the CPU tests; the local search and the merge are passed in,
so the same functions run over the oracle on CPU and over libfs.so on GPUs).
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


def shard_range(rank: int, world_size: int, nb: int) -> tuple[int, int]:
    """(first id, number of vectors) of a rank's database shard: contiguous, as even as possible,
    shard r below shard r + 1 (so that ties between shards keep ascending-id order)."""
    base, rem = divmod(nb, world_size)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def all_gather_lists(dist_local: torch.Tensor, ids_local: torch.Tensor) -> tuple[torch.Tensor, torch.Tensor]:
    """One all-gather of every rank's [nq, k] (distance fp32, id int64) lists -> [nq, G, k] each,
    shard g in slot g.  nq * k * 12 bytes per rank (12 MB at nq = 10^4, k = 100)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return dist_local[:, None, :].contiguous(), ids_local[:, None, :].contiguous()
    w = dist.get_world_size()
    nq, k = dist_local.shape
    # distances and ids travel in one buffer (the id as two 32-bit halves): one collective, not two
    packed = torch.empty((nq, k, 3), dtype=torch.int32, device=dist_local.device)
    packed[:, :, 0] = dist_local.contiguous().view(torch.int32)
    packed[:, :, 1:] = ids_local.contiguous().view(torch.int32).view(nq, k, 2)
    out = torch.empty((w * nq, k, 3), dtype=torch.int32, device=dist_local.device)  # rank-major concatenation
    dist.all_gather_into_tensor(out, packed)
    out = out.view(w, nq, k, 3)
    d = out[..., 0].contiguous().view(torch.float32).permute(1, 0, 2).contiguous()
    i = out[..., 1:].contiguous().view(torch.int64).view(w, nq, k).permute(1, 0, 2).contiguous()
    return d, i


def sharded_search(search_local, merge, id_base: int):
    """Database sharding: run `search_local()` -> (dist [nq, k], ids [nq, k], ids local to the shard,
    -1 = padding), make the ids global (+ id_base), exchange with one all-gather and merge with
    `merge(dist [nq, G, k], ids [nq, G, k]) -> (dist [nq, k], ids [nq, k])`.  Every rank returns the
    full result."""
    d, i = search_local()
    i = torch.where(i >= 0, i + id_base, i)
    dg, ig = all_gather_lists(d, i)
    return merge(dg, ig)
