"""Multi-GPU plumbing: rays are independent, so the path shards with no
data-path collective.  One process per GPU, ``torch.distributed`` (NCCL on GPUs, gloo in the CPU tests).

Two ways to use N ranks:
  * frames  (weak scaling, what ``bench.py --gpus N`` times): rank r renders frames r, r+N, ... of a movie;
  * tiles   (strong scaling of one image): ``raptor_set_shard(rank, world)`` makes the kernel take the 8x4-pixel
    tiles r, r+N, ... ; the ranks' zero-initialised images are summed (disjoint support => exact).
This module holds only index bookkeeping and the two reductions around the timed region.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

TILE_X, TILE_Y = 8, 4      # must match k_render's tile shape


def n_tiles(nx: int, ny: int) -> int:
    return ((nx + TILE_X - 1) // TILE_X) * ((ny + TILE_Y - 1) // TILE_Y)


def tiles_of_rank(nx: int, ny: int, rank: int, world: int) -> range:
    """Global tile indices (row-major) traced by ``rank`` after raptor_set_shard(rank, world)."""
    return range(rank, n_tiles(nx, ny), world)


def pixel_owner_map(nx: int, ny: int, world: int) -> torch.Tensor:
    """[ny, nx] int32: which rank traces each pixel under the tile sharding."""
    ntx = (nx + TILE_X - 1) // TILE_X
    iy, ix = torch.meshgrid(torch.arange(ny), torch.arange(nx), indexing="ij")
    tile = (iy // TILE_Y) * ntx + ix // TILE_X
    return (tile % world).to(torch.int32)


def frames_of_rank(n_frames: int, rank: int, world: int) -> range:
    return range(rank, n_frames, world)


def aggregate(elapsed_ms: float, units: float, device="cpu"):
    """(max over ranks of the time, sum over ranks of the units): the bench contract's whole-job numbers."""
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return t.item(), u.item()


def combine_tile_shards(image: torch.Tensor) -> torch.Tensor:
    """Sum of the ranks' images (each zero outside its own tiles): the full image on every rank."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(image, op=dist.ReduceOp.SUM)
    return image
