"""Shared helpers of the parity tests (no method arithmetic of either side)."""
import math

import numpy as np

DELTA_B = 0.05     # [M] half-width of the excluded band around the analytic critical curve (A20)


def critical_curve_points(a, incl_deg, n=4000):
    """Image-plane critical curve (shadow edge) of a Kerr hole, Bardeen (1973), with the paper's
    camera convention L = -alpha sin i: alpha_c = -xi/sin i, beta_c = +-sqrt(eta + a^2 cos^2 i - xi^2 cot^2 i)."""
    i = math.radians(incl_deg)
    if a == 0.0:
        t = np.linspace(0, 2 * math.pi, n)
        return math.sqrt(27.0) * np.cos(t), math.sqrt(27.0) * np.sin(t)
    r_pro = 2 * (1 + math.cos(2 / 3 * math.acos(-abs(a))))
    r_ret = 2 * (1 + math.cos(2 / 3 * math.acos(abs(a))))
    rs = np.linspace(r_pro, r_ret, n)
    xi = -(rs ** 3 - 3 * rs ** 2 + a * a * rs + a * a) / (a * (rs - 1))
    eta = rs ** 3 * (4 * a * a - rs * (rs - 3) ** 2) / (a * a * (rs - 1) ** 2)
    rad = eta + (a * math.cos(i)) ** 2 - xi ** 2 / math.tan(i) ** 2
    ok = rad >= 0
    al = -xi[ok] / math.sin(i)
    be = np.sqrt(rad[ok])
    return np.concatenate([al, al[::-1]]), np.concatenate([be, -be[::-1]])


def ring_mask(scene, delta_b=DELTA_B):
    """True for pixels whose centre lies within delta_b of the critical curve (photon-ring band)."""
    ca, cb = critical_curve_points(scene.a, scene.incl_deg)
    ax = (np.arange(scene.nx) + 0.5) * scene.fov_M / scene.nx - scene.fov_M / 2
    by = (np.arange(scene.ny) + 0.5) * scene.fov_M / scene.ny - scene.fov_M / 2
    A, B = np.meshgrid(ax, by)
    mask = np.zeros(A.shape, dtype=bool)
    # only pixels near the curve's bounding box need the distance
    near = (A > ca.min() - 1) & (A < ca.max() + 1) & (B > cb.min() - 1) & (B < cb.max() + 1)
    idx = np.argwhere(near)
    if idx.size:
        pa, pb = A[near], B[near]
        d2 = np.full(pa.shape, np.inf)
        for s in range(0, ca.size, 500):
            d = (pa[:, None] - ca[None, s:s + 500]) ** 2 + (pb[:, None] - cb[None, s:s + 500]) ** 2
            d2 = np.minimum(d2, d.min(1))
        mask[near] = d2 < delta_b ** 2
    return mask


def rel_err(gpu, ref):
    """|g - o| / max(|o|, 1e-30 max|o|) per pixel, per frequency plane (A20)."""
    gpu, ref = np.asarray(gpu, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    floor = 1e-30 * np.abs(ref).reshape(ref.shape[0], -1).max(1)
    floor = np.where(floor > 0, floor, 1e-300)
    return np.abs(gpu - ref) / np.maximum(np.abs(ref), floor[:, None, None])


def parity_report(scene, gpu, ref, delta_b=DELTA_B):
    """gpu/ref: dict(image [nf,ny,nx], status, nsteps).  Returns a dict of the parity numbers."""
    ring = ring_mask(scene, delta_b)
    err = rel_err(gpu["image"], ref["image"])
    keep = ~ring
    e = err[:, keep]
    return dict(
        n_excluded=int(ring.sum()),
        frac_ok=float((e <= 1e-8).mean()),
        max_err=float(e.max()),
        median_err=float(np.median(e)),
        status_equal=bool((gpu["status"][keep] == ref["status"][keep]).all()),
        nsteps_equal_frac=float((gpu["nsteps"][keep] == ref["nsteps"][keep]).mean()),
    )
