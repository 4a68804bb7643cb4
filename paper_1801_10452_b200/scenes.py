"""Seeded synthetic scenes: the INPUTS of the RAPTOR hot path (data, not algorithm).

This module serves both the CUDA path and the CPU oracle with the same numbers. It holds
none of the method's arithmetic (no metric, no connection, no camera, no transfer): only
the problem statement of each configuration (spin, camera distance and inclination, field
of view, pixel count, frequencies, plasma model constants -- PAPER.md:146-160, Table 2
PAPER.md:324-338, Table B.1) and the seeded GRMHD-like grids that stand
in for the BHAC / HARM2D dumps of the paper, which are not available.

It imports neither the CUDA binding nor anything under ``oracle/``.

Configurations C0..C4 are BASELINE.json ``configs[0..4]``; the recipe is stated in
DESIGN.md ("Input recipe") and follows SURVEY.md section 8(d).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

# --- CGS literals used to state the physical scale of a scene (data).  The CUDA path and
# --- the oracle each carry their own copy of the constants they compute with.
C_CGS = 2.99792458e10
G_CGS = 6.6743e-8
MSUN_G = 1.98841e33
PC_CM = 3.0856775814913673e18
M_P_G = 1.67262192e-24
M_E_G = 9.1093837e-28

# plasma_model codes (same numbering on both sides of the C ABI, include/raptor.h)
VACUUM, SPHERE, TORUS, GRID2D, GRID3DT, SLAB, DISK = 0, 1, 2, 3, 4, 5, 6
# grid_dtype codes
F64, F32 = 0, 1


@dataclass
class Scene:
    """Plain description of one rendering problem; field names follow ``raptor_params``."""
    name: str = "scene"
    # spacetime + chart (A.7-A.13 PAPER.md:585-605)
    a: float = 0.0
    mks_h: float = 1.0          # h = 1  => logarithmic Kerr-Schild
    mks_r0: float = 0.0
    mass: float = 1.0           # mass parameter m multiplying every "2r" (m = 0: flat space, tests)
    # camera (Eq. 25-29)
    r_cam: float = 1000.0
    incl_deg: float = 60.0
    fov_M: float = 40.0
    t_cam: float = 0.0
    nx: int = 64
    ny: int = 64
    # physical scaling (Table 2)
    M_bh_g: float = 4.5e6 * MSUN_G
    D_src_cm: float = 8.5e3 * PC_CM
    M_unit_g: float = 0.0       # rho0 = M_unit / L^3 (grid models)
    # integrator (Eq. 7-16; step rule: BASELINE.json configs[0] / Eq. 21-24)
    integrator: int = 0         # 0 = RK4
    step_policy: int = 0        # 0 = A: h = clamp(c (r - r_H), min, max); 1 = B: Eq. 21-24
    step_c: float = 0.05
    step_min: float = 1e-3
    step_max: float = 1.0
    eps: float = 0.03
    delta: float = 1e-40
    eps_polar: float = 0.125    # policy A polar guard: h <= eps_polar * r |sin theta|
    max_steps: int = 200000
    r_stop_in_factor: float = 1.01
    r_stop_out_factor: float = 1.1
    tau_cutoff: float = math.inf
    # frequencies [Hz]
    freq_hz: tuple = (230e9,)
    # plasma
    plasma_model: int = VACUUM
    model: tuple = (0.0,) * 16
    k2_mode: int = 0
    tp_over_te: float = 3.0
    te_model: int = 0           # 0: constant T_p/T_e; 1: Eq. 47 with model[0] = R_low, model[1] = R_high (grids)
    gamma_ad: float = 4.0 / 3.0
    # grid (models GRID2D, GRID3DT): AoS [t][i1][i2][i3][8] = rho,u,u~1,u~2,u~3,B1,B2,B3
    n1: int = 0
    n2: int = 0
    n3: int = 1
    nt: int = 1
    grid_dtype: int = F64
    slow_light: int = 0
    snapshot: int = 0           # fast light: which snapshot of a GRID3DT series is used
    precision: int = 0          # 0 = FP64 (the contract); 1 = FP32 (the paper's performance configuration only, Table B.1)
    x1_min: float = 0.0
    x1_max: float = 0.0
    t0: float = 0.0
    dt_snap: float = 1.0
    grid: Optional[np.ndarray] = field(default=None, repr=False)

    @property
    def n_freq(self) -> int:
        return len(self.freq_hz)

    @property
    def L_cm(self) -> float:
        return G_CGS * self.M_bh_g / C_CGS ** 2

    def with_pixels(self, nx: int, ny: Optional[int] = None) -> "Scene":
        return replace(self, nx=int(nx), ny=int(nx if ny is None else ny))


# ----------------------------------------------------------------------------------------
# counter-based RNG of the grid recipe: splitmix64, u = (z >> 11) * 2^-53
# ----------------------------------------------------------------------------------------
_M64 = (1 << 64) - 1


class SplitMix64:
    def __init__(self, seed: int):
        self.s = seed & _M64

    def next_u64(self) -> int:
        self.s = (self.s + 0x9E3779B97F4A7C15) & _M64
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
        return z ^ (z >> 31)

    def uniform(self) -> float:
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)

    def randint(self, lo: int, hi: int) -> int:
        """integer in [lo, hi] inclusive"""
        return lo + int(self.uniform() * (hi - lo + 1))


def draw_modes(seed: int, three_d: bool, n_fields: int = 8, n_modes: int = 16):
    """Mode table of the turbulent modulation, drawn in the fixed order
    (field, mode, p, q, s, w, psi, A).  2-D grids force s = w = 0 (the draws still happen)."""
    rng = SplitMix64(seed)
    table = np.zeros((n_fields, n_modes, 6))
    for f in range(n_fields):
        for m in range(n_modes):
            p = rng.randint(1, 6)
            q = rng.randint(1, 6)
            s = rng.randint(0, 4)
            w = rng.randint(-3, 3)
            psi = 2.0 * math.pi * rng.uniform()
            A = (0.5 + 0.5 * rng.uniform()) / n_modes
            if not three_d:
                s, w = 0, 0
            table[f, m] = (p, q, s, w, psi, A)
    return table


def _theta_of_x2(x2, h):
    return np.pi * x2 + 0.5 * (1.0 - h) * np.sin(2.0 * np.pi * x2)


def synthetic_grid(seed: int, a: float, h: float, n1: int, n2: int, n3: int = 1, nt: int = 1,
                   r_in: float = 1.2, r_out: float = 50.0, dt_snap: float = 10.0,
                   tp_over_te: float = 3.0, gamma_ad: float = 4.0 / 3.0,
                   dtype=np.float64) -> np.ndarray:
    """GRMHD-like primitives on a cell-centred MKS(h) grid, shape [nt, n1, n2, n3, 8].

    Fields: rho, u, u~^1, u~^2, u~^3, B^1, B^2, B^3 (HARM primitive ordering, PAPER.md:164,
    373): a torus plus tenuous atmosphere, each field modulated by (1 + 0.3 * sum of 16
    seeded smooth Fourier modes), tapered to exactly zero between r = 40 and r = 48.
    Everything is continuous in all coordinates and periodic in phi.
    """
    three_d = (n3 > 1) or (nt > 1)
    modes = draw_modes(seed, three_d)
    x1_min, x1_max = math.log(r_in), math.log(r_out)
    d1 = (x1_max - x1_min) / n1
    x1 = x1_min + (np.arange(n1) + 0.5) * d1
    x2 = (np.arange(n2) + 0.5) / n2
    ph = (np.arange(n3) + 0.5) * (2.0 * np.pi / n3)
    tt = np.arange(nt) * dt_snap
    xi1 = (x1 - x1_min) / (x1_max - x1_min)
    T_total = nt * dt_snap

    def delta(fidx):
        acc = np.zeros((nt, n1, n2, n3))
        for (p, q, s, w, psi, A) in modes[fidx]:
            e1 = np.exp(1j * 2.0 * np.pi * p * xi1)
            e2 = np.exp(1j * 2.0 * np.pi * q * x2)
            e3 = np.exp(1j * s * ph)
            e4 = np.exp(1j * (2.0 * np.pi * w * tt / T_total + psi))
            # Re( e4 (x) e1 (x) e2 (x) e3 ) = cos(2pi(p xi1 + q x2) + s phi + 2pi w t/T + psi)
            e12 = (e1[:, None] * e2[None, :])                    # [n1,n2]
            e34 = (e4[:, None] * e3[None, :])                    # [nt,n3]
            acc += A * (e34[:, None, None, :] * e12[None, :, :, None]).real
        return acc

    r = np.exp(x1)[None, :, None, None]
    th = _theta_of_x2(x2, h)[None, None, :, None]
    dth = (np.pi * (1.0 + (1.0 - h) * np.cos(2.0 * np.pi * x2)))[None, None, :, None]
    sth, cth = np.sin(th), np.cos(th)

    u_ = np.clip((r - 40.0) / 8.0, 0.0, 1.0)
    W = 1.0 - u_ * u_ * (3.0 - 2.0 * u_)
    bump = np.clip(1.0 - ((r - 12.0) / 8.0) ** 2, 0.0, None) ** 2

    out = np.empty((nt, n1, n2, n3, 8), dtype=dtype)
    rho = W * (bump * np.exp(-cth * cth / 0.18) + 1e-3 * r ** -1.5) * (1.0 + 0.3 * delta(0))
    theta_t = (120.0 / r) * (1.0 + 0.3 * delta(1))
    uu = rho * theta_t * (M_E_G / M_P_G) * (1.0 + tp_over_te) / (gamma_ad - 1.0)
    out[..., 0] = rho
    out[..., 1] = uu
    out[..., 2] = -0.05 * r ** -1.5 * (1.0 + 0.3 * delta(2))
    out[..., 3] = 0.02 * r ** -1.5 * delta(3) / dth
    out[..., 4] = (1.0 + 0.3 * delta(4)) / (r ** 1.5 + a)
    # field strength from beta_p = 10 with flat-space-like scale factors (a data recipe)
    b2 = 2.0 * (gamma_ad - 1.0) * uu / 10.0
    sb = np.sqrt(b2)
    out[..., 5] = 0.2 * sb / r * delta(5)
    out[..., 6] = 0.2 * sb / (r * dth) * delta(6)
    out[..., 7] = sb / (r * sth) * (1.0 + 0.3 * delta(7))
    return out


# ----------------------------------------------------------------------------------------
# the five configurations of BASELINE.json
# ----------------------------------------------------------------------------------------
_A_KERR = 0.9375
_L_CM_SGRA = G_CGS * 4.5e6 * MSUN_G / C_CGS ** 2
# rho = 1 (code) <-> n_e = 1e7 cm^-3
_M_UNIT_GRID = 1e7 * (M_P_G + M_E_G) * _L_CM_SGRA ** 3

_grid_cache: dict = {}


def _cached_grid(key, **kw):
    if key not in _grid_cache:
        _grid_cache[key] = synthetic_grid(**kw)
    return _grid_cache[key]


def config_C0(nx: int = 64) -> Scene:
    """Schwarzschild, analytic optically thin sphere (BASELINE.json configs[0])."""
    # model = [n0, n_exp, T0, T_exp, beta]
    return Scene(name="C0", a=0.0, mks_h=1.0, incl_deg=60.0, nx=nx, ny=nx,
                 plasma_model=SPHERE,
                 model=(1e6, -1.5, 1e11, -1.0, 10.0) + (0.0,) * 11)


def config_C1(nx: int = 512) -> Scene:
    """Kerr a=0.9375, analytic torus (BASELINE.json configs[1])."""
    # model = [n_max, r_peak, r_halfwidth, scale_height, T0, T_exp, beta]
    return Scene(name="C1", a=_A_KERR, mks_h=1.0, incl_deg=60.0, nx=nx, ny=nx,
                 plasma_model=TORUS,
                 model=(1e7, 12.0, 8.0, 0.3, 1e11, -1.0, 10.0) + (0.0,) * 9)


def config_C2(nx: int = 1024, n1: int = 256, n2: int = 256) -> Scene:
    """Kerr, 2-D axisymmetric seeded grid, fast light (BASELINE.json configs[2])."""
    g = _cached_grid(("2d", n1, n2), seed=1801, a=_A_KERR, h=0.3, n1=n1, n2=n2)
    return Scene(name="C2", a=_A_KERR, mks_h=0.3, incl_deg=20.0, nx=nx, ny=nx,
                 plasma_model=GRID2D, M_unit_g=_M_UNIT_GRID,
                 n1=n1, n2=n2, n3=1, nt=1, grid_dtype=F64,
                 x1_min=math.log(1.2), x1_max=math.log(50.0), grid=g[0])


def config_C3(nx: int = 256, n_freq: int = 32, n1: int = 256, n2: int = 256) -> Scene:
    """Spectrum: C2's grid, 32 log-spaced frequencies 1e9..1e16 Hz (BASELINE.json configs[3])."""
    s = config_C2(nx=nx, n1=n1, n2=n2)
    if n_freq > 1:
        nu = tuple(1e9 * 10.0 ** (7.0 * k / (n_freq - 1)) for k in range(n_freq))
    else:
        nu = (230e9,)
    return replace(s, name="C3", freq_hz=nu)


def light_travel_offset(r_cam: float, r_ref: float = 10.0) -> float:
    """Coordinate-time offset between a camera at r_cam and radius r_ref along the outgoing radial null ray of
    ingoing Kerr-Schild Schwarzschild, t(r) = r + 4 ln(r - 2) + const.  The ONE home of
    this formula: a number attached to a scene (t_cam) or to a snapshot window, not part of the method."""
    return (r_cam + 4.0 * math.log(r_cam - 2.0)) - (r_ref + 4.0 * math.log(r_ref - 2.0))


def slow_light_t_cam(r_cam: float, t_mid: float) -> float:
    """Camera time that centres the snapshot window on t_mid: replaces the paper's empirical
    calibration as a first guess; raptor_calibrate_delay refines it from two light curves."""
    return t_mid + light_travel_offset(r_cam)


def config_C4(nx: int = 1024, n1: int = 128, n2: int = 64, n3: int = 64, nt: int = 32,
              slow_light: bool = True) -> Scene:
    """Slow light through a 3-D + time seeded grid in float32 (BASELINE.json configs[4]);
    ``slow_light=False`` gives the fast-light image of the middle snapshot."""
    g = _cached_grid(("3dt", n1, n2, n3, nt), seed=10452, a=_A_KERR, h=0.3,
                     n1=n1, n2=n2, n3=n3, nt=nt, dt_snap=10.0, dtype=np.float32)
    mid = nt // 2
    t_mid = mid * 10.0
    return Scene(name="C4" if slow_light else "C4-fast", a=_A_KERR, mks_h=0.3, incl_deg=60.0,
                 nx=nx, ny=nx, t_cam=slow_light_t_cam(1000.0, t_mid) if slow_light else 0.0,
                 plasma_model=GRID3DT, M_unit_g=_M_UNIT_GRID,
                 n1=n1, n2=n2, n3=n3, nt=nt, grid_dtype=F32,
                 slow_light=1 if slow_light else 0, snapshot=mid,
                 x1_min=math.log(1.2), x1_max=math.log(50.0), t0=0.0, dt_snap=10.0, grid=g)


def slab_scene(n_e: float, theta_e: float, B_gauss: float, thickness_M: float,
               sin_pitch: float = 1.0, nu_hz: float = 230e9, nx: int = 4, **kw) -> Scene:
    """Test scene: flat space (mass parameter 0), static uniform slab |z| < thickness/2.
    model = [n_e, Theta_e, B, half_thickness, sin(pitch angle)]"""
    base = dict(name="slab", a=0.0, mass=0.0, mks_h=1.0, incl_deg=30.0, r_cam=200.0, fov_M=10.0,
                nx=nx, ny=nx, plasma_model=SLAB, freq_hz=(nu_hz,),
                model=(n_e, theta_e, B_gauss, 0.5 * thickness_M, sin_pitch) + (0.0,) * 11,
                r_stop_in_factor=1.01, r_stop_out_factor=1.1)
    base.update(kw)
    return Scene(**base)


def config_PB1(nx: int = 512, n1: int = 256, n2: int = 256) -> Scene:
    """The paper's own performance configuration (Table B.1): 512 x 512 pixels, image size 40 M,
    step rule Eq. 21-24 with eps = 0.03, integration scheme "RK2" (midpoint [A17]), radiative transfer on; camera,
    frequency, inclination, tau cut-off and T_p/T_e from Table 2: r_cam = 1e4 M, 230 GHz,
    i = 90 deg, tau_cutoff = ln 1000, T_p/T_e = 3.  The BHAC dump is replaced by the seeded 2-D grid of C2; FP64
    instead of the paper's single precision."""
    base = config_C2(nx=nx, n1=n1, n2=n2)
    return replace(base, name="PB1", incl_deg=90.0, r_cam=1.0e4, integrator=3, step_policy=1, eps=0.03,
                   tau_cutoff=math.log(1000.0), tp_over_te=3.0)


def thin_disk(a: float = 0.0, incl_deg: float = 60.0, nx: int = 256, r_out: float = 15.0, max_order: int = 10,
              p: float = 3.0, r_in: float = 0.0, **kw) -> Scene:
    """Thin-disk workload of Sect. 4.2.1: equatorial Keplerian disk from the ISCO (r_in <= 0)
    to 15 M, emission coefficient ~ 1/r^2, no absorption; lensed images up to ``max_order`` (Fig. 5: 10; the line
    spectra of Fig. 6 use 1).  model = [r_in, r_out, max_order, p]"""
    base = dict(name="thin_disk", a=a, mks_h=1.0, incl_deg=incl_deg, r_cam=1000.0, fov_M=40.0, nx=nx, ny=nx,
                plasma_model=DISK, model=(r_in, r_out, float(max_order), p) + (0.0,) * 12)
    base.update(kw)
    return Scene(**base)


def config_PB1_f32(nx: int = 512, n1: int = 256, n2: int = 256) -> Scene:
    """PB1 in the paper's own precision (Table B.1: "Single precision: yes")."""
    return replace(config_PB1(nx=nx, n1=n1, n2=n2), name="PB1F32", precision=1)


CONFIGS = {"C0": config_C0, "C1": config_C1, "C2": config_C2, "C3": config_C3, "C4": config_C4, "PB1": config_PB1, "PB1F32": config_PB1_f32}


def config(name: str, **kw) -> Scene:
    return CONFIGS[name](**kw)
