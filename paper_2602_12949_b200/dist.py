"""Host-side multi-GPU plumbing of the benchmark: the path shards by texels with the
model replicated and NO data-path collective, so all that is distributed is (a) the parameter blob, broadcast once from
rank 0, (b) which frame -- or which rows of the one frame -- a rank owns and (c) the max-over-ranks of the device time.
torch.distributed only (nccl on GPUs, gloo in the CPU tests)."""
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


def row_range_of_rank(height: int, rank: int, world: int, rows_per_tile: int = 4) -> tuple:
    """Strong-scaling split of ONE image for niv_infer_image: contiguous blocks of whole 4-row tile rows (SURVEY 8(e):
    "contiguous row-blocks of the frame per GPU")."""
    tiles = (height + rows_per_tile - 1) // rows_per_tile
    lo = (tiles * rank) // world * rows_per_tile
    hi = min(height, (tiles * (rank + 1)) // world * rows_per_tile)
    return lo, hi


def broadcast_params(arrays, shapes_dtypes, device, src: int = 0):
    """The model is replicated: rank `src` holds the parameter blobs as numpy arrays (`arrays`: a list, None elsewhere),
    every rank gets them as tensors on `device` through ONE broadcast per blob ("ncclBroadcast of the
    parameter blob once").  shapes_dtypes: [(shape, torch dtype)] -- known to every rank from the model spec."""
    import torch
    import torch.distributed as dist
    out = []
    world = dist.get_world_size() if (dist.is_available() and dist.is_initialized()) else 1
    rank = dist.get_rank() if world > 1 else src
    for k, (shape, dtype) in enumerate(shapes_dtypes):
        if rank == src:
            t = torch.from_numpy(arrays[k]).reshape(shape).to(device=device, dtype=dtype)
        else:
            t = torch.empty(shape, dtype=dtype, device=device)
        if world > 1:
            dist.broadcast(t, src=src)
        out.append(t)
    return out


def launcher_command(n_ranks: int, port: int, script: str, argv: list) -> list:
    """`python bench.py --gpus N` outside torchrun starts its own ranks: one process per GPU on this node."""
    import sys
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n_ranks),
            "--master-addr", "127.0.0.1", "--master-port", str(port), script] + list(argv)
