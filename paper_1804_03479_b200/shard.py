"""Multi-GPU plumbing of the patch-group update: none of it touches the data path.

Patch groups are independent inside mhd_advance (all coupling goes through the ghost zones the caller filled,
PAPER.md:234-236), so N GPUs = N processes that each advance their own contiguous range of groups; the only
cross-rank values are one scalar MAX for the CFL time step and, in bench.py, the MAX of the device
times.  torch.distributed (NCCL on GPUs, gloo in the CPU tests) carries those scalars.
"""
from __future__ import annotations


def shard_range(ngroups: int, rank: int, world: int):
    """Contiguous, balanced range [first, first + count) of rank `rank` out of `world` (sizes differ by at most 1)."""
    if world < 1 or not (0 <= rank < world) or ngroups < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(ngroups, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX of a per-rank scalar (device time of the timed region, max signal speed of the local groups)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def global_dt(local_max_speed: float, dh: float, cfl: float, dist=None, device="cpu") -> float:
    """CFL step of the whole job from each rank's mhd_dt_reduce max speed (R13): cfl * dh / max over ranks."""
    return cfl * dh / max_over_ranks(local_max_speed, dist, device)
