"""ctypes front end of the CPU oracle (oracle/raptor_oracle.c).  TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from the CUDA
package; a scene is any object carrying the attributes of ``raptor_params`` (duck-typed),
normally a ``paper_1801_10452_b200.scenes.Scene`` built by the caller.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "raptor_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_LIB_F32 = os.path.join(_HERE, "liboracle_f32.so")

STATUS = {0: "RUNNING", 1: "CAPTURED", 2: "ESCAPED", 3: "MAXSTEPS", 4: "THICK", 5: "NONFINITE"}


def build(force: bool = False, dtype: str = "f64") -> str:
    """gcc -O2 -ffp-contract=off (no FMA contraction) -fopenmp, rows-only parallelism.  dtype "f32": the SAME source
    with real = float and single-precision constants (Table B.1 of the paper: "Single precision: yes")."""
    out = _LIB if dtype == "f64" else _LIB_F32
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-Wall", "-shared", "-fPIC"]
        if dtype == "f32":
            cmd += ["-DORC_REAL=float", "-fsingle-precision-constant"]
        subprocess.check_call(cmd + ["-o", out, _SRC, "-lm"])
    return out


class _Types:
    """ctypes mirror of the oracle's types for one working precision (real = double or float)."""

    def __init__(self, dtype: str):
        assert dtype in ("f64", "f32"), dtype
        self.dtype = dtype
        R = self.REAL = C.c_double if dtype == "f64" else C.c_float
        self.np_real = np.float64 if dtype == "f64" else np.float32
        self.D4 = R * 4
        self.D44 = (R * 4) * 4
        self.D444 = ((R * 4) * 4) * 4

        class OrcParams(C.Structure):
            _fields_ = [
                ("a", R), ("mks_h", R), ("mks_r0", R), ("mass", R),
                ("r_cam", R), ("incl_deg", R), ("fov_M", R), ("t_cam", R),
                ("M_bh_g", C.c_double), ("D_src_cm", C.c_double), ("M_unit_g", C.c_double),     # beyond float range
                ("step_c", R), ("step_min", R), ("step_max", R),
                ("eps", R), ("delta", R), ("eps_polar", R),
                ("r_stop_in_factor", R), ("r_stop_out_factor", R), ("tau_cutoff", R),
                ("model", R * 16),
                ("tp_over_te", R), ("gamma_ad", R),
                ("x1_min", R), ("x1_max", R), ("t0", R), ("dt_snap", R),
                ("freq_hz", C.POINTER(R)),
                ("grid", C.c_void_p),
                ("nx", C.c_int32), ("ny", C.c_int32), ("integrator", C.c_int32), ("step_policy", C.c_int32),
                ("max_steps", C.c_int32), ("n_freq", C.c_int32), ("plasma_model", C.c_int32), ("k2_mode", C.c_int32),
                ("n1", C.c_int32), ("n2", C.c_int32), ("n3", C.c_int32), ("nt", C.c_int32),
                ("grid_dtype", C.c_int32), ("slow_light", C.c_int32), ("snapshot", C.c_int32), ("te_model", C.c_int32),
            ]

        class RayResult(C.Structure):
            _fields_ = [("status", C.c_int32), ("nsteps", C.c_int32), ("nsampled", C.c_int32), ("pad_", C.c_int32),
                        ("null_max", R), ("X", R * 4), ("K", R * 4)]

        self.OrcParams, self.RayResult = OrcParams, RayResult
        L = self.lib = C.CDLL(build(dtype=dtype))
        L.orc_sizeof_params.restype = C.c_size_t
        L.orc_sizeof_ray_result.restype = C.c_size_t
        assert L.orc_sizeof_params() == C.sizeof(OrcParams), (L.orc_sizeof_params(), C.sizeof(OrcParams))
        assert L.orc_sizeof_ray_result() == C.sizeof(RayResult)
        PP, D4, D44 = C.POINTER(OrcParams), self.D4, self.D44
        L.orc_null_norm.restype = R
        L.orc_step_size.restype = R
        L.orc_planck.restype = R
        L.orc_planck.argtypes = [R, R]
        L.orc_emissivity.restype = R
        L.orc_emissivity.argtypes = [R] * 5 + [C.c_int]
        L.orc_bessel_k2.restype = R
        L.orc_bessel_k2.argtypes = [R]
        L.orc_horizon.restype = R
        L.orc_r_isco.restype = R
        L.orc_r_isco.argtypes = [R]
        L.orc_line_profile.argtypes = [PP, C.c_void_p, C.c_void_p, C.c_int, R, R, C.c_void_p]
        L.orc_transfer_update.argtypes = [C.POINTER(R), C.POINTER(R)] + [R] * 5
        L.orc_mks_theta.argtypes = [R, R] + [C.POINTER(R)] * 3
        L.orc_x2_of_theta.argtypes = [R, R, R, C.POINTER(R)]
        L.orc_metric_ks.argtypes = [R] * 4 + [D44]
        L.orc_metric_ks_inv.argtypes = [R] * 4 + [D44]
        L.orc_camera_ab.argtypes = [PP, R, R, D4, D4]
        L.orc_pixel_ab.argtypes = [PP, C.c_int, C.c_int, C.POINTER(R), C.POINTER(R)]
        L.orc_rk4_step.argtypes = [PP, D4, D4, R]
        L.orc_verlet_step.argtypes = [PP, D4, D4, R, C.c_int]
        L.orc_rk2_step.argtypes = [PP, D4, D4, R]
        L.orc_step.argtypes = [PP, D4, D4, R]
        L.orc_transfer.argtypes = [PP, D4, D4, R, C.c_void_p, C.c_void_p]
        L.orc_calibrate_delay.restype = R
        L.orc_calibrate_delay.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, R, C.c_int, C.POINTER(R)]
        L.orc_trace_ray.argtypes = [PP, R, R, C.c_void_p, C.c_void_p, C.POINTER(RayResult), C.c_void_p, C.c_int, C.c_int]


_types: dict = {}


def types(dtype: str = "f64") -> _Types:
    if dtype not in _types:
        _types[dtype] = _Types(dtype)
    return _types[dtype]


def lib(dtype: str = "f64"):
    return types(dtype).lib


# the float64 structures under their old names
def __getattr__(name):
    if name in ("OrcParams", "RayResult"):
        return getattr(types("f64"), name)
    raise AttributeError(name)


class Oracle:
    """Holds an ``orc_params`` built from a scene and keeps the arrays it points at alive."""

    def __init__(self, scene, dtype: str = "f64"):
        """dtype "f32": the single-precision build of the same source (8(f) f1, Table B.1 of the paper)."""
        self.scene = scene
        self.T = T = types(dtype)
        p = T.OrcParams()
        for name in ("a", "mks_h", "mks_r0", "mass", "r_cam", "incl_deg", "fov_M", "t_cam", "M_bh_g",
                     "D_src_cm", "M_unit_g", "step_c", "step_min", "step_max", "eps", "delta", "eps_polar",
                     "r_stop_in_factor", "r_stop_out_factor", "tau_cutoff", "tp_over_te", "gamma_ad",
                     "x1_min", "x1_max", "t0", "dt_snap"):
            setattr(p, name, float(getattr(scene, name)))
        for name in ("nx", "ny", "integrator", "step_policy", "max_steps", "plasma_model", "k2_mode",
                     "n1", "n2", "n3", "nt", "grid_dtype", "slow_light", "snapshot", "te_model"):
            setattr(p, name, int(getattr(scene, name)))
        m = list(scene.model) + [0.0] * (16 - len(scene.model))
        p.model = (T.REAL * 16)(*m[:16])
        self._freq = np.ascontiguousarray(np.asarray(scene.freq_hz, dtype=T.np_real))
        p.n_freq = int(self._freq.size)
        p.freq_hz = self._freq.ctypes.data_as(C.POINTER(T.REAL))
        self._grid = None
        if getattr(scene, "grid", None) is not None:
            want = np.float32 if scene.grid_dtype == 1 else np.float64
            self._grid = np.ascontiguousarray(scene.grid, dtype=want)
            expect = scene.nt * scene.n1 * scene.n2 * scene.n3 * 8
            assert self._grid.size == expect, (self._grid.shape, expect)
            p.grid = self._grid.ctypes.data
        self.p = p
        self.lib = T.lib

    # ---- geometry -------------------------------------------------------------------
    @property
    def r_horizon(self) -> float:
        return self.lib.orc_horizon(C.byref(self.p))

    def metric(self, X):
        g = self.T.D44()
        self.lib.orc_metric_mks(C.byref(self.p), self.T.D4(*X), g)
        return np.array(g)

    def metric_inv(self, X):
        g = self.T.D44()
        self.lib.orc_metric_mks_inv(C.byref(self.p), self.T.D4(*X), g)
        return np.array(g)

    def dmetric(self, X):
        dg = self.T.D444()
        self.lib.orc_dmetric_mks(C.byref(self.p), self.T.D4(*X), dg)
        return np.array(dg)

    def christoffel(self, X):
        G = self.T.D444()
        self.lib.orc_christoffel_mks(C.byref(self.p), self.T.D4(*X), G)
        return np.array(G)

    def rhs(self, X, K):
        f = self.T.D4()
        self.lib.orc_rhs(C.byref(self.p), self.T.D4(*X), self.T.D4(*K), f)
        return np.array(f)

    def null_norm(self, X, K) -> float:
        return self.lib.orc_null_norm(C.byref(self.p), self.T.D4(*X), self.T.D4(*K))

    def conserved(self, X, K):
        E, L, Q = self.T.REAL(), self.T.REAL(), self.T.REAL()
        self.lib.orc_conserved(C.byref(self.p), self.T.D4(*X), self.T.D4(*K), C.byref(E), C.byref(L), C.byref(Q))
        return E.value, L.value, Q.value

    def camera(self, alpha, beta):
        X, K = self.T.D4(), self.T.D4()
        self.lib.orc_camera_ab(C.byref(self.p), float(alpha), float(beta), X, K)
        return np.array(X), np.array(K)

    def pixel_ab(self, ix, iy):
        al, be = self.T.REAL(), self.T.REAL()
        self.lib.orc_pixel_ab(C.byref(self.p), int(ix), int(iy), C.byref(al), C.byref(be))
        return al.value, be.value

    def step_size(self, X, K) -> float:
        return self.lib.orc_step_size(C.byref(self.p), self.T.D4(*X), self.T.D4(*K))

    def rk4_step(self, X, K, dl):
        Xc, Kc = self.T.D4(*X), self.T.D4(*K)
        self.lib.orc_rk4_step(C.byref(self.p), Xc, Kc, float(dl))
        return np.array(Xc), np.array(Kc)

    def verlet_step(self, X, K, dl, corrector=False):
        Xc, Kc = self.T.D4(*X), self.T.D4(*K)
        self.lib.orc_verlet_step(C.byref(self.p), Xc, Kc, float(dl), 1 if corrector else 0)
        return np.array(Xc), np.array(Kc)

    def rk2_step(self, X, K, dl):
        Xc, Kc = self.T.D4(*X), self.T.D4(*K)
        self.lib.orc_rk2_step(C.byref(self.p), Xc, Kc, float(dl))
        return np.array(Xc), np.array(Kc)

    def step(self, X, K, dl):
        """One step of the scene's integrator (0 RK4, 1 Verlet, 2 Verlet + corrector, 3 RK2)."""
        Xc, Kc = self.T.D4(*X), self.T.D4(*K)
        self.lib.orc_step(C.byref(self.p), Xc, Kc, float(dl))
        return np.array(Xc), np.array(Kc)

    # ---- plasma + transfer ----------------------------------------------------------
    def grid_interp(self, X):
        prim = (self.T.REAL * 8)()
        ok = self.lib.orc_grid_interp(C.byref(self.p), self.T.D4(*X), prim)
        return (np.array(prim) if ok else None)

    def plasma(self, X):
        ne, th, B, sf = self.T.REAL(), self.T.REAL(), self.T.REAL(), self.T.REAL()
        u, p = self.T.D4(), self.T.D4()
        ok = self.lib.orc_plasma(C.byref(self.p), self.T.D4(*X), C.byref(ne), C.byref(th), C.byref(B), u, p, C.byref(sf))
        if not ok:
            return None
        return dict(n_e=ne.value, theta_e=th.value, B=B.value, u=np.array(u), p=np.array(p), sin_fixed=sf.value)

    def transfer(self, X, K, h, I, tau):
        I = np.ascontiguousarray(I, dtype=self.T.np_real).copy()
        tau = np.ascontiguousarray(tau, dtype=self.T.np_real).copy()
        ok = self.lib.orc_transfer(C.byref(self.p), self.T.D4(*X), self.T.D4(*K), self.T.REAL(h),
                                   I.ctypes.data_as(C.c_void_p), tau.ctypes.data_as(C.c_void_p))
        return ok, I, tau

    # ---- rays and images ------------------------------------------------------------
    def trace(self, alpha, beta, record_path: bool = False, monitor_null: bool = False, max_path: int = 400000):
        nf = self.p.n_freq
        I = np.zeros(nf, dtype=self.T.np_real)
        tau = np.zeros(nf, dtype=self.T.np_real)
        res = self.T.RayResult()
        path = None
        if record_path:
            path = np.zeros((max_path, 8), dtype=self.T.np_real)
        self.lib.orc_trace_ray(C.byref(self.p), float(alpha), float(beta), I.ctypes.data, tau.ctypes.data,
                               C.byref(res), path.ctypes.data if path is not None else None,
                               max_path if path is not None else 0, 1 if monitor_null else 0)
        out = dict(I=I, tau=tau, status=res.status, nsteps=res.nsteps, nsampled=res.nsampled,
                   null_max=res.null_max, X=np.array(res.X), K=np.array(res.K))
        if path is not None:
            out["path"] = path[:min(res.nsteps, max_path)]
        return out

    def render_disk(self):
        """Thin-disk workload: dict(image = sum of g^p/r^2 over counted crossings, redshift = g of the first one)."""
        p = self.p
        image = np.zeros((1, p.ny, p.nx), dtype=self.T.np_real)
        red = np.zeros((1, p.ny, p.nx), dtype=self.T.np_real)
        status = np.zeros((p.ny, p.nx), dtype=np.int32)
        nsteps = np.zeros((p.ny, p.nx), dtype=np.int32)
        steps, sampled = C.c_uint64(), C.c_uint64()
        self.lib.orc_render_rows2(C.byref(p), image.ctypes.data_as(C.c_void_p), red.ctypes.data_as(C.c_void_p),
                                  status.ctypes.data_as(C.c_void_p), nsteps.ctypes.data_as(C.c_void_p), 0, int(p.ny), 1,
                                  C.byref(steps), C.byref(sampled))
        return dict(image=image, redshift=red, status=status, nsteps=nsteps, steps=steps.value, sampled=sampled.value)

    def line_profile(self, image_I, image_g, nbins, g_min, g_max):
        a = np.ascontiguousarray(image_I, dtype=self.T.np_real)
        b = np.ascontiguousarray(image_g, dtype=self.T.np_real)
        hist = np.zeros(int(nbins), dtype=self.T.np_real)
        self.lib.orc_line_profile(C.byref(self.p), a.ctypes.data_as(C.c_void_p), b.ctypes.data_as(C.c_void_p), int(nbins),
                                  float(g_min), float(g_max), hist.ctypes.data_as(C.c_void_p))
        return hist

    def render(self, rows=None, row_stride: int = 1):
        """Full image (or rows [row0,row1) with a stride).  Returns dict(image, status, nsteps, steps, sampled)."""
        p = self.p
        image = np.zeros((p.n_freq, p.ny, p.nx), dtype=self.T.np_real)
        status = np.zeros((p.ny, p.nx), dtype=np.int32)
        nsteps = np.zeros((p.ny, p.nx), dtype=np.int32)
        steps, sampled = C.c_uint64(), C.c_uint64()
        r0, r1 = (0, p.ny) if rows is None else rows
        self.lib.orc_render_rows(C.byref(p), image.ctypes.data_as(C.c_void_p), status.ctypes.data_as(C.c_void_p),
                                 nsteps.ctypes.data_as(C.c_void_p), int(r0), int(r1), int(row_stride),
                                 C.byref(steps), C.byref(sampled))
        return dict(image=image, status=status, nsteps=nsteps, steps=steps.value, sampled=sampled.value)

    def flux(self, image):
        image = np.ascontiguousarray(image, dtype=self.T.np_real)
        out = np.zeros(self.p.n_freq, dtype=self.T.np_real)
        self.lib.orc_flux(C.byref(self.p), image.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p))
        return out


# free functions -----------------------------------------------------------------------
def planck(nu, theta_e, dtype="f64"):
    return lib(dtype).orc_planck(float(nu), float(theta_e))


def emissivity(nu, n_e, theta_e, B, sin_th, k2_mode=0, dtype="f64"):
    return lib(dtype).orc_emissivity(float(nu), float(n_e), float(theta_e), float(B), float(sin_th), int(k2_mode))


def r_isco(a, dtype="f64"):
    return lib(dtype).orc_r_isco(float(a))


def bessel_k2(x, dtype="f64"):
    return lib(dtype).orc_bessel_k2(float(x))


def transfer_update(I, tau, j, alpha, nu_hat, Lcm, h, dtype="f64"):
    T = types(dtype)
    Ic, tc = T.REAL(I), T.REAL(tau)
    T.lib.orc_transfer_update(C.byref(Ic), C.byref(tc), j, alpha, nu_hat, Lcm, h)
    return Ic.value, tc.value


def mks_theta(h, x2, dtype="f64"):
    T = types(dtype)
    th, d1, d2 = T.REAL(), T.REAL(), T.REAL()
    T.lib.orc_mks_theta(float(h), float(x2), C.byref(th), C.byref(d1), C.byref(d2))
    return th.value, d1.value, d2.value


def x2_of_theta(h, theta, tol=1e-15, dtype="f64"):
    T = types(dtype)
    x2 = T.REAL()
    it = T.lib.orc_x2_of_theta(float(h), float(theta), float(tol), C.byref(x2))
    return x2.value, it


def metric_ks(a, m, r, th, dtype="f64"):
    T = types(dtype)
    g = T.D44()
    T.lib.orc_metric_ks(float(a), float(m), float(r), float(th), g)
    return np.array(g)


def metric_ks_inv(a, m, r, th, dtype="f64"):
    T = types(dtype)
    g = T.D44()
    T.lib.orc_metric_ks_inv(float(a), float(m), float(r), float(th), g)
    return np.array(g)


def calibrate_delay(t_fast, F_fast, t_slow, F_slow, max_shift, n_grid=2001, dtype="f64"):
    """Sect. 5.1: (delay, rms) -- the oracle's plain grid search."""
    T = types(dtype)
    arr = [np.ascontiguousarray(x, dtype=T.np_real) for x in (t_fast, F_fast, t_slow, F_slow)]
    rms = T.REAL()
    d = T.lib.orc_calibrate_delay(arr[0].size, arr[0].ctypes.data, arr[1].ctypes.data, arr[2].size, arr[2].ctypes.data,
                                  arr[3].ctypes.data, float(max_shift), int(n_grid), C.byref(rms))
    return d, rms.value
