"""Host-side multi-GPU plumbing of the benchmark: the path shards by texels with the model
replicated and NO data-path collective, so all that is distributed is (a) which frame a rank owns and (b) the
max-over-ranks of the device time.  torch.distributed only (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import os


def env_rank_world():
    """(rank, world_size, local_rank) from the torchrun environment (1-process defaults)."""
    def _i(name, default):
        try:
            return int(os.environ.get(name, default))
        except ValueError:
            return default
    return _i("RANK", 0), _i("WORLD_SIZE", 1), _i("LOCAL_RANK", 0)


def frame_of_rank(rank: int, world: int, step_frames: int = 1) -> list:
    """Frames (camera sub-seeds) owned by `rank`: weak scaling, `step_frames` whole frames per rank per step."""
    if not 0 <= rank < world:
        raise ValueError("rank %d outside world of %d" % (rank, world))
    return [rank * step_frames + k for k in range(step_frames)]


def texel_range_of_rank(n: int, rank: int, world: int, tile: int = 128) -> tuple:
    """Strong-scaling split of ONE frame of n texels: contiguous ranges of whole 128-texel tiles."""
    tiles = (n + tile - 1) // tile
    lo = (tiles * rank) // world * tile
    hi = min(n, (tiles * (rank + 1)) // world * tile)
    return lo, hi


def reduce_max(value: float, device=None) -> float:
    """Max over ranks of a host float (the timed region's device milliseconds)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gqps(texels_per_rank: int, world: int, ms_per_step_max: float) -> float:
    """Aggregate throughput of all ranks in Gqueries/s from the max-over-ranks step time."""
    return world * texels_per_rank / (ms_per_step_max * 1e-3) / 1e9
