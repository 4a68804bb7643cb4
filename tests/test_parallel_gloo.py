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
        # the exact function bench.py --scaling strong times, with a fake renderer standing in for raptor_render
        # under raptor_set_shard(rank, world): it writes this rank's tiles only and leaves the rest untouched
        calls = []

        def fake_render_shard(img):
            assert float(img.abs().sum()) == 0.0            # strong_step zeroed it first
            img[owner == rank] = full[owner == rank]
            calls.append("render")

        def fake_flux(img):
            calls.append("flux")
            return img.sum()

        stale = torch.full_like(full, 99.0)                 # last step's image: must not leak into this one
        flux = parallel.strong_step(fake_render_shard, stale, fake_flux)
        strong_ok = bool(torch.equal(stale, full)) and float(flux) == float(full.sum()) and calls == ["render", "flux"]
        assert parallel.world_info() == (rank, world)
        out.put((rank, bool(torch.equal(combined, full)) and strong_ok, t, u, frames))
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


def test_owner_map_is_the_raster_tile_index_mod_world():
    # raptor_set_shard(rank, world): tile (tx, ty) of the 8x4-pixel tiling belongs to rank (ty * ntx + tx) % world
    nx, ny, world = 52, 38, 3
    owner = parallel.pixel_owner_map(nx, ny, world)
    ntx, nty = 7, 10
    for ty in range(nty):
        for tx in range(ntx):
            assert int(owner[min(4 * ty, ny - 1), 8 * tx]) == (ty * ntx + tx) % world
            assert int(owner[min(4 * ty + 3, ny - 1), min(8 * tx + 7, nx - 1)]) == (ty * ntx + tx) % world


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


def test_frame_of_rank_gives_every_rank_its_own_frame():
    from paper_1801_10452_b200 import scenes
    c4 = scenes.config_C4(nx=8, n1=8, n2=8, n3=4, nt=4)
    ts = [parallel.frame_of_rank(c4, r).t_cam for r in range(4)]
    assert ts[0] == c4.t_cam and all(b - a == 2.5 for a, b in zip(ts, ts[1:]))          # own camera time
    c2 = scenes.config_C2(nx=8, n1=16, n2=16)
    g = [parallel.frame_of_rank(c2, r).grid for r in range(3)]
    assert g[0] is c2.grid and g[1].shape == c2.grid.shape
    assert not (g[1] == g[0]).all() and not (g[2] == g[1]).all() and (g[1][..., 0] > 0).all()   # own seeded snapshot
    fast = scenes.config_C4(nx=8, n1=8, n2=8, n3=4, nt=4, slow_light=False)
    assert [parallel.frame_of_rank(fast, r).snapshot for r in range(3)] == [2, 3, 0]
    c1 = scenes.config_C1(8)
    assert parallel.frame_of_rank(c1, 3) is c1                                          # stationary analytic scene
