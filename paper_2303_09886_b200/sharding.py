"""Multi-GPU layout of the path: antennas are independent, so they shard across ranks with the
weights replicated and no data-path collective.  Host logic only."""
from __future__ import annotations


def shard_antennas(n_antennas: int, world: int, rank: int) -> range:
    """Contiguous block of antennas owned by `rank`; blocks differ in size by at most one."""
    if world < 1 or not (0 <= rank < world) or n_antennas < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(n_antennas, world)
    start = rank * base + min(rank, extra)
    return range(start, start + base + (1 if rank < extra else 0))


def rank_slice(world: int, rank: int, packed, coarse, fine_delay, phase, gains) -> dict:
    """What one rank builds its engine from: the contiguous antenna block of every per-antenna array (antenna is the
    outermost index of all of them and of in / out, include/fengine.h), plus `n_antennas` and the block itself.
    The weights are replicated, not sliced."""
    import numpy as np
    block = shard_antennas(int(packed.shape[0]), world, rank)
    sl = slice(block.start, block.stop)
    for name, arr in (("coarse", coarse), ("fine_delay", fine_delay), ("phase", phase), ("gains", gains)):
        if arr.shape[0] != packed.shape[0]:
            raise ValueError(f"{name}: antenna must be the outermost index")
    return dict(n_antennas=len(block), antennas=block, packed=np.ascontiguousarray(packed[sl]),
                coarse=np.ascontiguousarray(coarse[sl]), fine_delay=np.ascontiguousarray(fine_delay[sl]),
                phase=np.ascontiguousarray(phase[sl]), gains=np.ascontiguousarray(gains[sl]))


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """Max of a timing scalar over the ranks of the default process group (the only collective of the job)."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: int, world: int, seconds_max: float) -> float:
    """Whole-job throughput: units all ranks processed / slowest rank's time (weak scaling)."""
    return world * units_per_rank / seconds_max
