"""Multi-GPU sharding of a workloads.Config.  Ions are independent
 and seeding is counter-based on the global ion index, so a rank only needs its
index range; the single exchange step is the sum of the integer counters."""
from __future__ import annotations

import copy


def shard_config(cfg, rank: int, world: int, mode: str = "weak"):
    """Per-rank copy of `cfg`.
    weak  : every rank traces cfg.n_ions ions of its own (first_index += rank * 2^40);
    strong: each group's ions are split into `world` contiguous index ranges."""
    out = copy.copy(cfg)
    out.groups = []
    for g in cfg.groups:
        h = copy.copy(g)
        if mode == "weak":
            h.first_index = g.first_index + (rank << 40)
        elif mode == "strong":
            lo = (g.n_ions * rank) // world
            hi = (g.n_ions * (rank + 1)) // world
            h.first_index, h.n_ions = g.first_index + lo, hi - lo
        else:
            raise ValueError(mode)
        out.groups.append(h)
    return out


def allreduce_counters(dist, *tensors):
    """Sum the per-rank integer histograms / summaries in place (NCCL on GPUs, gloo on CPU)."""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        for t in tensors:
            dist.all_reduce(t)
