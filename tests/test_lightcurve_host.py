"""Host logic of light curves / slow-light movies: sliding snapshot window, frame sharding
over ranks (world-size-2 gloo on CPU), time calibration of Sect. 5.1.  No GPU."""
import math
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1801_10452_b200 import lightcurve as lc


def test_window_start_centres_on_the_departure_time_and_clips():
    nt, n_snap, dt = 8, 100, 10.0
    off = lc.light_travel_offset(1000.0)
    assert off == 1000.0 + 4 * math.log(998.0) - 10.0 - 4 * math.log(8.0)      # t(r) = r + 4 ln(r - 2)  [A15]
    # light that left r = 10 M at t = 500 reaches the camera at t_cam = 500 + off: window centred on snapshot 50
    lo = lc.window_start(500.0 + off, 1000.0, 0.0, dt, nt, n_snap)
    assert lo <= 50 <= lo + nt - 1 and abs((lo + 0.5 * (nt - 1)) - 50.0) <= 0.5
    assert lc.window_start(-1e6, 1000.0, 0.0, dt, nt, n_snap) == 0
    assert lc.window_start(1e6, 1000.0, 0.0, dt, nt, n_snap) == n_snap - nt
    # monotone in t_cam
    los = [lc.window_start(t + off, 1000.0, 0.0, dt, nt, n_snap) for t in np.linspace(0, 990, 200)]
    assert all(b >= a for a, b in zip(los, los[1:]))


def test_window_streamer_uploads_only_new_snapshots_into_their_slots():
    nt = 4
    slots, log = {}, []

    def upload(m, arr):
        assert arr == ("snap", m)
        slots[m % nt] = m
        log.append(m)

    windows = []
    ws = lc.WindowStreamer(nt, lambda m: ("snap", m), upload, windows.append, resident=range(nt))
    for m in range(nt):
        slots[m] = m
    assert ws.move_to(0) == 0 and log == []
    assert ws.move_to(1) == 1 and log == [4] and slots == {0: 4, 1: 1, 2: 2, 3: 3}
    assert ws.move_to(3) == 2 and log == [4, 5, 6]
    assert ws.move_to(10) == 4 and sorted(slots.values()) == [10, 11, 12, 13]
    for s, m in slots.items():
        assert m % nt == s
    assert ws.move_to(9) == 1 and log[-1] == 9          # moving back re-uploads the one that was overwritten
    assert windows == [0, 1, 3, 10, 9] and ws.uploads == 8


def test_calibrate_delay_recovers_a_known_shift():
    # Sect. 5.1: the slow-light curve is the fast-light curve translated on the time axis.  The ORACLE's
    # grid search is pinned by a known shift; the library's host routine (raptor_calibrate_delay, reached through
    # lightcurve.calibrate_delay; no GPU involved) must then agree with the oracle.
    from oracle import oracle as orc
    t = np.arange(0.0, 2000.0, 10.0)
    f = lambda x: 2.0 + 0.4 * np.sin(x / 90.0) + 0.2 * np.sin(x / 37.0 + 1.0) + 0.1 * np.cos(x / 11.0)
    for true in (-63.0, 0.0, 41.5):
        do, ro = orc.calibrate_delay(t, f(t), t, 3.0 * f(t - true), max_shift=150.0, n_grid=3001)
        assert abs(do - true) <= 0.5 and ro < 2e-2, (do, ro)     # residual: linear interpolation between samples
        d, rms = lc.calibrate_delay(t, f(t), t, 3.0 * f(t - true), max_shift=150.0, n_grid=3001)
        assert d == pytest.approx(do, abs=1e-9) and rms == pytest.approx(ro, rel=1e-9)
    # by hand: two-point "curves" -- fast (t = 0, 1; F = 1, 3), slow = the same line shifted by +0.25 in time
    ts = np.array([-1.0, 0.0, 1.0, 2.0])
    Fs = 1.0 + 2.0 * (ts - 0.25)
    tf, Ff = np.array([0.0, 0.5, 1.0, 1.5]), 1.0 + 2.0 * np.array([0.0, 0.5, 1.0, 1.5])
    # unnormalised the match would be exact at d = 0.25; the means differ, so check the oracle against numpy instead
    grid = np.linspace(-0.5, 0.5, 101)
    rms_np = [np.sqrt(np.mean((np.interp(tf + d, ts, Fs) / Fs.mean() - Ff / Ff.mean()) ** 2)) for d in grid]
    do, ro = orc.calibrate_delay(tf, Ff, ts, Fs, 0.5, 101)
    assert do == pytest.approx(grid[int(np.argmin(rms_np))], abs=1e-12) and ro == pytest.approx(min(rms_np), rel=1e-10)
    # a shift that leaves fewer than max(4, n/2) points is skipped; nothing qualifies -> rms = inf
    assert orc.calibrate_delay(tf, Ff, ts + 100.0, Fs, 0.5, 11)[1] == math.inf
    assert lc.calibrate_delay(tf, Ff, ts + 100.0, Fs, 0.5, 11) == (0.0, math.inf)


def test_calibrate_delay_refuses_curves_it_cannot_normalise_or_interpolate():
    # a zero mean would normalise to inf/nan and a time axis that is not ascending has no interpolation interval:
    # both used to come back as (0, inf) "no shift qualified"; now they are errors with a message
    from paper_1801_10452_b200 import binding
    t = np.linspace(0.0, 10.0, 21)
    F = 1.0 + 0.1 * np.sin(t)
    zero_mean = np.array([1.0, -1.0] * 10 + [0.0])
    for args in ((t, zero_mean, t, F), (t, F, t, np.zeros_like(F)), (t, F, t[::-1].copy(), F),
                 (t, F, np.concatenate([t[:5], t[4:-1]]), F)):
        with pytest.raises(binding.RaptorError) as err:
            binding.raptor_calibrate_delay(*args, 1.0, 11)
        assert err.value.code == binding.EINVAL and "raptor_calibrate_delay" in str(err.value)
    assert binding.raptor_calibrate_delay(t, F, t, 2.0 * F, 1.0, 11)[0] == 0.0


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_frames, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank "renders" all frames with garbage in the rows it does not own; the gather keeps the owners' rows
        full = torch.arange(n_frames * 3, dtype=torch.float64).reshape(n_frames, 3) + 1.0
        mine = full + 1000.0 * (rank + 1)
        for f in lc.frames_of_rank(n_frames, rank, world):
            mine[f] = full[f]
        got = lc.combine_frame_shards(mine, n_frames, rank, world)
        out.put((rank, bool(torch.equal(got, full)), list(lc.frames_of_rank(n_frames, rank, world))))
    finally:
        dist.destroy_process_group()


def test_two_rank_frame_sharding_gathers_the_whole_curve():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    world, n_frames, port = 2, 7, _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_frames, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _ in results)
    assert sorted(results[0][2] + results[1][2]) == list(range(n_frames))
