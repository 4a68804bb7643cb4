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
    """Tiles (raster index ty * ntx + tx) traced by ``rank`` after raptor_set_shard(rank, world): those whose index is
    rank mod world.  The kernel launches them nearest to the image centre first; the order does not change the image."""
    return range(rank, n_tiles(nx, ny), world)


def pixel_owner_map(nx: int, ny: int, world: int) -> torch.Tensor:
    """[ny, nx] int32: which rank traces each pixel under the tile sharding."""
    ntx = (nx + TILE_X - 1) // TILE_X
    iy, ix = torch.meshgrid(torch.arange(ny), torch.arange(nx), indexing="ij")
    return (((iy // TILE_Y) * ntx + ix // TILE_X) % world).to(torch.int32)


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


def world_info():
    """(rank, world) of the initialised process group, (0, 1) without one."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def frame_of_rank(scene, rank: int, frame_dt: float = 2.5, seed_stride: int = 1):
    """Weak scaling = a movie, one frame per rank: a slow-light scene gets its own camera time
    t_cam + rank * frame_dt, a fast-light grid scene its own snapshot (the seeded generator with seed + rank), an
    analytic scene is stationary (every frame is the same image).  Pure bookkeeping on the scene description."""
    from dataclasses import replace
    if rank == 0:
        return scene
    if getattr(scene, "slow_light", 0):
        return replace(scene, t_cam=scene.t_cam + rank * frame_dt)
    if getattr(scene, "grid", None) is not None and scene.nt == 1 and scene.n3 == 1:
        from . import scenes
        g = scenes.synthetic_grid(seed=1801 + seed_stride * rank, a=scene.a, h=scene.mks_h, n1=scene.n1, n2=scene.n2)
        return replace(scene, grid=g[0])
    if getattr(scene, "grid", None) is not None:
        return replace(scene, snapshot=(scene.snapshot + rank) % scene.nt)
    return scene


def strong_step(render_shard, image: torch.Tensor, reduce_flux):
    """One strong-scaling step of ONE image over all ranks: every rank traces its interleaved
    tiles (raptor_set_shard(rank, world) was called on its context) into a zeroed image, one all-reduce(SUM) of the
    image makes it whole on every rank (disjoint support: exact), and the flux is reduced from the whole image.
    ``render_shard(image)`` and ``reduce_flux(image)`` are the two C-ABI calls; this function is what
    ``bench.py --scaling strong`` times and what the world-size-2 gloo test drives with a fake renderer."""
    image.zero_()
    render_shard(image)
    combine_tile_shards(image)
    return reduce_flux(image)
