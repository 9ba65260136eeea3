"""Multi-GPU sharding: simulations are independent, so plans are partitioned
across ranks with NO data-path collective; graph, tables and (if used) the request stream are
replicated. The only exchange is a gather of the per-plan results at the end (kilobytes)."""
from __future__ import annotations

from typing import Tuple

import numpy as np
import torch
import torch.distributed as dist


def plan_shard(n_plans: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced [begin, end) range of plans owned by `rank` (keeps a plan's rates,
    trials and bisection steps on one GPU)."""
    base, rem = divmod(n_plans, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def shard_workload(w, rank: int, world: int):
    """The slice of a workloads.Workload this rank evaluates."""
    import copy
    b, e = plan_shard(w.plans.n_plans, rank, world)
    idx = np.arange(b, e)
    s = copy.copy(w)
    s.plans = w.plans.subset(idx)
    if w.rate_mrps is not None:
        s.rate_mrps = w.rate_mrps[idx]
    if w.rate_hi_mrps is not None:
        s.rate_hi_mrps = w.rate_hi_mrps[idx]
    if w.plan_variant is not None:
        s.plan_variant = w.plan_variant[idx]
    return s, idx


def gather_plan_results(local: torch.Tensor, n_plans: int) -> torch.Tensor:
    """All-gather per-plan results (first dim = this rank's plans, in plan_shard order) into the
    full [n_plans, ...] tensor on every rank. Works with NCCL (CUDA tensors) and gloo (CPU)."""
    if not dist.is_initialized() or dist.get_world_size() == 1:
        return local
    world = dist.get_world_size()
    sizes = [plan_shard(n_plans, r, world) for r in range(world)]
    longest = max(e - b for b, e in sizes)
    pad = torch.zeros((longest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([parts[r][: e - b] for r, (b, e) in enumerate(sizes)], dim=0)


def best_plan(goodput_mrps: torch.Tensor) -> int:
    """Default selection policy: arg-max of goodput summed over types (Algorithm 2 l.17,
    PAPER.md:258). Ties resolve to the lowest plan index."""
    total = goodput_mrps.to(torch.int64).sum(dim=1)
    return int(torch.argmax(total).item())
