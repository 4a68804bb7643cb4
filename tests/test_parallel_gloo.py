"""N > 1 host logic on CPU: world-size-2 gloo processes exercise the tile/frame bookkeeping and the two
reductions bench.py performs around its timed region (max of the time, sum of the units, sum of the shards)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1801_10452_b200 import parallel


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nx, ny, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank "renders" its own tiles into a zero image: pixel value = 1 + global pixel index
        owner = parallel.pixel_owner_map(nx, ny, world)
        full = (1 + torch.arange(nx * ny, dtype=torch.float64)).reshape(ny, nx)
        mine = torch.where(owner == rank, full, torch.zeros_like(full))
        combined = parallel.combine_tile_shards(mine.clone())
        t, u = parallel.aggregate(10.0 + rank, float((owner == rank).sum()))
        frames = list(parallel.frames_of_rank(7, rank, world))
        out.put((rank, bool(torch.equal(combined, full)), t, u, frames))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_and_aggregation():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    nx, ny, world = 52, 38, 2
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, nx, ny, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ok, t, u, frames in results:
        assert ok                                   # disjoint shards sum to the full image exactly
        assert t == 11.0 and u == nx * ny           # max over ranks of the time, sum over ranks of the units
    assert sorted(results[0][4] + results[1][4]) == list(range(7))


def test_tiles_are_dealt_exactly_once():
    for nx, ny, world in [(52, 38, 2), (1024, 1024, 8), (9, 5, 4), (1, 1, 3)]:
        seen = []
        for r in range(world):
            seen += list(parallel.tiles_of_rank(nx, ny, r, world))
        assert sorted(seen) == list(range(parallel.n_tiles(nx, ny)))
        owner = parallel.pixel_owner_map(nx, ny, world)
        assert owner.shape == (ny, nx) and int(owner.max()) < world
        counts = torch.bincount(owner.flatten(), minlength=world)
        if parallel.n_tiles(nx, ny) >= 4 * world:
            assert counts.max() - counts.min() <= 2 * 32 + nx     # balanced to within a couple of tiles / ragged edge
