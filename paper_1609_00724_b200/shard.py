"""Multi-GPU plumbing: field lines are independent, so the path shards over ranks with no data-path
collective.  The field is replicated on every rank; each rank traces a contiguous range of the seed array (seed arrays
of the configs are lattice-ordered, so a contiguous range is spatially compact) and the per-seed outputs concatenate.
Only orchestration lives here: torch.distributed for the plumbing, every computation is a libqsl call on the rank's GPU.
"""
from __future__ import annotations

import torch


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """[lo, hi) of the seeds rank `rank` traces: contiguous, disjoint, covering, sizes differing by at most one."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def gather_concat(local: torch.Tensor, n_total: int, group=None) -> torch.Tensor:
    """All-gathers the per-seed output of every rank's shard (first dimension = seeds of shard_range) into the full
    array in caller order, on every rank.  The one exchange a sharded level loop needs (L before FLEDGE)."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    base, rem = divmod(n_total, world)
    width = base + (1 if rem else 0)
    pad = torch.zeros((width,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    out = [parts[r][: shard_range(n_total, r, world)[1] - shard_range(n_total, r, world)[0]] for r in range(world)]
    return torch.cat(out, 0)


def reduce_job(ms_local: float, units_local: float, device="cpu", group=None) -> tuple[float, float]:
    """(max over ranks of the device time, sum over ranks of the units processed): the two reductions bench.py needs."""
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
        dist.all_reduce(u, op=dist.ReduceOp.SUM, group=group)
    return float(t.item()), float(u.item())
