"""Multi-GPU plumbing: runs are independent and keyed by their GLOBAL run index (O3), so a job
shards by run index with no data-path collective; the only exchanges are the max-over-ranks device time and an
optional final gather of per-run results (12-16 bytes per run).  torch.distributed (NCCL on GPUs, gloo in the
CPU tests) is plumbing only."""
from __future__ import annotations
import torch
import torch.distributed as dist


def shard_runs(total_runs: int, world: int, rank: int):
    """Contiguous, balanced partition of run indices [0, total_runs): -> (first_run, n_runs) of this rank."""
    base, rem = divmod(int(total_runs), int(world))
    n = base + (1 if rank < rem else 0)
    first = rank * base + min(rank, rem)
    return first, n


def max_over_ranks(value: float, device="cpu") -> float:
    """Device time of a multi-rank step = the slowest rank's."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: int, device="cpu") -> int:
    """Whole-job count of units (candidates) = the sum of every rank's."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return int(value)
    t = torch.tensor([int(value)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return int(t.item())


def gather_runs(local: torch.Tensor, total_runs: int) -> torch.Tensor | None:
    """Gathers per-run rows (n_local, k) of every rank into global run order on rank 0 (None elsewhere)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    world, rank = dist.get_world_size(), dist.get_rank()
    sizes = [shard_runs(total_runs, world, r)[1] for r in range(world)]
    pad = max(sizes)
    buf = torch.zeros((pad,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    buf[:local.shape[0]] = local
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    if rank != 0:
        return None
    return torch.cat([o[:n] for o, n in zip(out, sizes)], dim=0)
