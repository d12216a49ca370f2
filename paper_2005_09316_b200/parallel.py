"""Multi-GPU host logic.

Every visibility is independent (Eq 9 / Eq 11, sum over components only),
so the path shards by OUTPUT: each rank predicts a contiguous block of time steps with the
full (replicated, < 1 MB) component arrays.  There is no data-path collective.  The only
communication is (i) the max-over-ranks of the timed region and (ii), for a consumer that
wants one buffer, a single all-gather of disjoint shards.  One process per GPU;
`torch.distributed` (nccl on GPUs, gloo in the CPU tests) is plumbing only.

Nothing here computes visibilities.
"""
from __future__ import annotations

from typing import List, Optional

from . import inputs


def rank_workload(config: int, rank: int, world: int, *, scaling: str = "weak") -> inputs.Workload:
    """The Workload rank `rank` of `world` predicts.

    weak  : every rank gets the config's own T time steps of one observation that is `world`
            times longer (same array, same sky): per-GPU work is fixed (bench.py).
    strong: the config's T time steps are split contiguously over ranks (inputs.time_shard).
    """
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    if world == 1:
        return inputs.make_config(config)
    T = inputs.make_config_shape(config)[1]
    if scaling == "weak":
        return inputs.make_config(config, t_index0=rank * T, n_times=T, n_times_total=T * world)
    if scaling == "strong":
        t0, n = inputs.time_shard(T, rank, world)
        if n == 0:
            raise ValueError("more ranks than time steps")
        return inputs.make_config(config, t_index0=t0, n_times=n, n_times_total=T)
    raise ValueError("scaling must be 'weak' or 'strong'")


def max_over_ranks(value: float, dist=None, device: Optional[str] = None) -> float:
    """Max of a scalar over all ranks (timed regions are reported as the slowest rank's)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_time_shards(vis_local, dist=None) -> List:
    """All-gather of the ranks' [T_r, F, B] visibility shards (ragged in T allowed); returns
    the list ordered by rank, i.e. by time.  torch.cat(result) is the whole observation."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [vis_local]
    import torch
    world = dist.get_world_size()
    n_t = torch.tensor([vis_local.shape[0]], dtype=torch.int64, device=vis_local.device)
    counts = [torch.zeros_like(n_t) for _ in range(world)]
    dist.all_gather(counts, n_t)
    t_max = max(int(c.item()) for c in counts)
    pad = torch.zeros((t_max,) + tuple(vis_local.shape[1:]), dtype=vis_local.dtype, device=vis_local.device)
    pad[: vis_local.shape[0]] = vis_local
    # complex tensors travel as their real view (gloo has no complex all_gather)
    real = torch.view_as_real(pad) if pad.is_complex() else pad
    out = [torch.empty_like(real) for _ in range(world)]
    dist.all_gather(out, real.contiguous())
    res = []
    for c, o in zip(counts, out):
        o = torch.view_as_complex(o) if vis_local.is_complex() else o
        res.append(o[: int(c.item())])
    return res
