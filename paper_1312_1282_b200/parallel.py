"""Multi-GPU plumbing: walkers are independent Markov chains, so the path
shards by walker with NO data-path collective; the only exchange is the final reduction of a few
numbers per walker.  Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

from typing import Dict, Tuple

import torch
import torch.distributed as dist

from . import workloads as wl


def shard_for_rank(w: wl.Workload, rank: int, world: int) -> Tuple[list, int]:
    """(walkers_per_group, walker_id_base) of this rank's contiguous share of the workload's walkers
    (strong scaling of a fixed walker population; results are identical to the 1-GPU run because the
    global walker id keys each walker's random stream)."""
    begin, end = wl.walker_shard(w.n_walkers, rank, world)
    return wl.shard_groups(w, begin, end)


def walker_statistics(per_walker: torch.Tensor, group=None) -> Dict[str, torch.Tensor]:
    """Mean and standard error over ALL ranks' walkers of per-walker quantities [W_local][k]
    (one all_reduce of 2k+1 numbers)."""
    x = per_walker.to(torch.float64)
    k = x.shape[1]
    acc = torch.zeros(2 * k + 1, dtype=torch.float64, device=x.device)
    acc[:k] = x.sum(0)
    acc[k:2 * k] = (x * x).sum(0)
    acc[2 * k] = x.shape[0]
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(acc, op=dist.ReduceOp.SUM, group=group)
    n = acc[2 * k]
    mean = acc[:k] / n
    var = torch.clamp(acc[k:2 * k] / n - mean * mean, min=0.0) * n / torch.clamp(n - 1, min=1.0)
    return {"mean": mean, "se": torch.sqrt(var / n), "n": n}


def gather_walkers(per_walker: torch.Tensor, world_counts, group=None) -> torch.Tensor:
    """Concatenate per-walker rows of all ranks in global walker order (ranks own contiguous ranges)."""
    if not (dist.is_available() and dist.is_initialized()):
        return per_walker
    nmax = max(world_counts)                       # all_gather wants equal shapes: pad, then trim
    pad = torch.zeros((nmax,) + tuple(per_walker.shape[1:]), dtype=per_walker.dtype, device=per_walker.device)
    pad[:per_walker.shape[0]] = per_walker
    bufs = [torch.empty_like(pad) for _ in world_counts]
    dist.all_gather(bufs, pad, group=group)
    return torch.cat([b[:n] for b, n in zip(bufs, world_counts)], 0)
