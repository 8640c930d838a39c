"""Env sharding across ranks: envs are independent episodes (PAPER.md:556 runs them as
separate pool tasks), so each rank owns a contiguous env range and the data path has NO collective.
The only exchanges are the timing reduction (max over ranks) and, if a caller wants them, the per-env
results gathered at the end.  Backend-agnostic (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def env_range(rank: int, world_size: int, envs_per_rank: int):
    """Weak scaling: rank r owns global env ids [r*E, (r+1)*E)."""
    assert 0 <= rank < world_size and envs_per_rank > 0
    return rank * envs_per_rank, (rank + 1) * envs_per_rank


def split_envs(total_envs: int, world_size: int):
    """Strong-scaling split of a fixed batch: contiguous ranges, sizes differing by at most one."""
    base, rem = divmod(total_envs, world_size)
    out, lo = [], 0
    for r in range(world_size):
        n = base + (1 if r < rem else 0)
        out.append((lo, lo + n))
        lo += n
    return out


def max_over_ranks(x: float, device=None) -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: int, device=None) -> int:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return int(x)
    t = torch.tensor([x], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return int(t.item())


def gather_env_results(local: torch.Tensor) -> torch.Tensor:
    """Per-env results (flags, counters; a few bytes per env) of all ranks, concatenated in env order."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    parts = [torch.empty_like(local) for _ in range(dist.get_world_size())]
    dist.all_gather(parts, local.contiguous())
    return torch.cat(parts, dim=0)
