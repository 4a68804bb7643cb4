"""Light curves and slow-light movies (Sect. 5 of the paper).

Host-side bookkeeping only; every frame is rendered by the CUDA library through the C ABI
(``raptor_set_window`` / ``raptor_upload_snapshot`` / ``raptor_light_curve``).

* A series of n_snap snapshots (spacing dt_snap) longer than the context's nt slots is streamed through a
  sliding window: a frame with camera time t_cam needs the snapshots that cover the coordinate times its rays
  spend inside the grid, [t_cam - light_travel - depth, t_cam - light_travel + depth] ("the slices
  of GRMHD data should extend from the moment in time when the first ray enters the simulation volume until the
  moment when the last ray leaves it"); ``window_start`` centres the window on the arrival time of the frame.
* Frames are independent: with N ranks, rank r renders frames r, r + N, ... and the per-frame fluxes are
  gathered with one all_gather of n_frames x n_freq doubles; no data-path collective.
* Time calibration (Sect. 5.1): the delay that aligns a slow-light light curve with the fast-light
  one, found by minimising their mean squared difference over a shift of the time axis.
"""
from __future__ import annotations

import math
from typing import Callable, Sequence

import numpy as np


from .scenes import light_travel_offset      # [A15 in DESIGN.md]: one home, scenes.py


def window_start(t_cam: float, r_cam: float, t0: float, dt_snap: float, nt: int, n_snap: int) -> int:
    """First snapshot index of the nt-slot window for the frame with camera time t_cam: the window is centred on
    the time the frame's light left the inner region, clipped to the series [0, n_snap - nt]."""
    centre = (t_cam - light_travel_offset(r_cam) - t0) / dt_snap
    lo = int(math.floor(centre - 0.5 * (nt - 1) + 0.5))
    return max(0, min(lo, max(0, n_snap - nt)))


def frames_of_rank(n_frames: int, rank: int, world: int) -> range:
    return range(rank, n_frames, world)


class WindowStreamer:
    """Keeps a context's nt slots filled with the snapshots [lo, lo + nt) of a longer series, uploading only the
    snapshots that are new when the window moves.  ``get_snapshot(m)`` returns snapshot m as a host array
    [n1][n2][n3][8]; ``upload(m, array)`` and ``set_window(lo)`` are the two C-ABI calls (injected so that the
    logic is testable without a GPU)."""

    def __init__(self, nt: int, get_snapshot: Callable[[int], np.ndarray], upload: Callable[[int, np.ndarray], None],
                 set_window: Callable[[int], None], resident: Sequence[int] = ()):
        self.nt, self.get, self.upload, self.set_window = nt, get_snapshot, upload, set_window
        self.slots = {m % nt: m for m in resident}      # slot -> snapshot index held
        self.uploads = 0

    def move_to(self, lo: int) -> int:
        """Makes [lo, lo + nt) resident.  Returns the number of snapshots uploaded."""
        n = 0
        for m in range(lo, lo + self.nt):
            if self.slots.get(m % self.nt) != m:
                self.upload(m, self.get(m))
                self.slots[m % self.nt] = m
                n += 1
        self.set_window(lo)
        self.uploads += n
        return n


def render_light_curve(R, t_cams: Sequence[float], series=None, n_snap: int | None = None, rank: int = 0, world: int = 1):
    """Fluxes [n_frames][n_freq] (numpy, Jy) of the frames with camera times ``t_cams`` on ``R`` (a binding.Raptor of a
    slow-light GRID3DT scene).  ``series(m)`` returns snapshot m for series longer than the context's nt slots
    (None: the context's own nt snapshots are the whole series).  With world > 1 (torch.distributed initialised)
    every rank renders its share of the frames and all ranks return the full curve."""
    import torch
    import torch.distributed as dist

    s = R.scene
    n_frames = len(t_cams)
    out = torch.zeros((n_frames, R.nf), dtype=torch.float64, device="cuda")
    streamer = None
    if series is not None:
        streamer = WindowStreamer(s.nt, series, R.upload_snapshot, R.set_window, resident=range(s.nt))
    for f in frames_of_rank(n_frames, rank, world):
        if streamer is not None:
            streamer.move_to(window_start(t_cams[f], s.r_cam, s.t0, s.dt_snap, s.nt, n_snap))
        out[f] = R.light_curve(1, t_cams[f], 0.0)[0]
    if world > 1 and dist.is_available() and dist.is_initialized():
        dist.all_reduce(out, op=dist.ReduceOp.SUM)       # disjoint rows: the sum is the gather
    return out.cpu().numpy()


def combine_frame_shards(flux, n_frames: int, rank: int, world: int):
    """CPU-testable core of the gather: ``flux`` [n_frames][n_freq] holds this rank's frames (zeros elsewhere)."""
    import torch
    import torch.distributed as dist
    t = torch.as_tensor(flux, dtype=torch.float64).clone()
    mine = torch.zeros(n_frames, dtype=torch.bool)
    mine[list(frames_of_rank(n_frames, rank, world))] = True
    t[~mine] = 0.0
    if world > 1 and dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t


def calibrate_delay(t_fast, F_fast, t_slow, F_slow, max_shift: float, n_grid: int = 2001):
    """Sect. 5.1: the delay d for which F_slow(t + d) best matches F_fast(t) (least squares over the
    overlap, both curves normalised by their means), "effectively equivalent to translating the slow-light light
    curve with respect to the fast-light light curve on the time axis".  Returns (d, rms residual at d)."""
    from . import binding
    return binding.raptor_calibrate_delay(t_fast, F_fast, t_slow, F_slow, max_shift, n_grid)
