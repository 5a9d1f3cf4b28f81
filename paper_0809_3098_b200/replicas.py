"""Multi-GPU: replicas only.

The path does not shard profitably at the paper's sizes: a blocked whole-chip sweep of 1025^2 is ~1 us of
work and a time step has 1000 dependent ones, so any inter-GPU halo exchange would dominate.  What the paper
does run many of is independent Reynolds numbers on one grid (Table 1): one context per GPU, no
data-path collective.  This module holds the host logic: which Reynolds number a rank simulates and how
per-rank timings combine into the whole-job figure (max of the times, sum of the units).
"""
from dataclasses import replace

# Table 1 of the paper: Re of the six production runs on the 1024 x 1024 grid.
TABLE1_RE = (5000.0, 10000.0, 15000.0, 20000.0, 25000.0, 30000.0)


def replica_workload(base, rank: int, world: int):
    """Workload of `rank`: rank 0 keeps `base` (the config the metric is quoted on); the others take the
    same grid, dt, sweep count and relaxation factor at the next Reynolds numbers of Table 1 (cyclically),
    with their own seed.  Per-GPU work is identical: weak scaling."""
    if world <= 1 or rank == 0:
        return base
    ladder = [r for r in TABLE1_RE if r != base.Re]
    re = ladder[(rank - 1) % len(ladder)]
    return replace(base, name="%s_replica%d_Re%g" % (base.name, rank, re), Re=re, seed=base.seed + 1000 * rank)


def combine(units_local: float, seconds_local: float, world: int, dist=None, device=None):
    """(total units, max seconds) over the ranks.  `dist` is torch.distributed (initialised) or None."""
    if world <= 1 or dist is None:
        return units_local, seconds_local
    import torch
    t = torch.tensor([seconds_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()), float(t.item())
