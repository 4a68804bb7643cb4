"""Thin ctypes binding of include/raptor.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of ``libraptor_b200.so``; PyTorch is used for
device memory and streams.  There is no CPU fallback: if the library is missing, import of the
library handle raises.  Function names mirror the C ABI (``raptor_create`` ... ``raptor_destroy``);
``Raptor`` is a small RAII convenience around them.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libraptor_b200.so")
ABI_VERSION = 3
MAX_FREQ = 64

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED = 0, -1, -2, -3, -4
STATUS = {0: "RUNNING", 1: "CAPTURED", 2: "ESCAPED", 3: "MAXSTEPS", 4: "THICK", 5: "NONFINITE"}

# every symbol include/raptor.h declares
SYMBOLS = ("raptor_create", "raptor_upload_grid", "raptor_set_shard", "raptor_render", "raptor_render_disk",
           "raptor_line_profile", "raptor_set_camera_time", "raptor_set_window", "raptor_upload_snapshot",
           "raptor_light_curve", "raptor_calibrate_delay", "raptor_spectrum", "raptor_flux", "raptor_flux_static",
           "raptor_render_host", "raptor_trace", "raptor_eval_rhs", "raptor_null_norm", "raptor_set_null_monitor", "raptor_get_counters", "raptor_fp64_peak", "raptor_fp32_peak", "raptor_fp64_probe",
           "raptor_destroy", "raptor_last_error")


class RaptorParams(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("abi_version", C.c_uint32),
        ("a", C.c_double), ("mks_h", C.c_double), ("mks_r0", C.c_double), ("mass", C.c_double),
        ("r_cam", C.c_double), ("incl_deg", C.c_double), ("fov_M", C.c_double), ("t_cam", C.c_double),
        ("M_bh_g", C.c_double), ("D_src_cm", C.c_double), ("M_unit_g", C.c_double),
        ("step_c", C.c_double), ("step_min", C.c_double), ("step_max", C.c_double),
        ("eps", C.c_double), ("delta", C.c_double), ("eps_polar", C.c_double),
        ("r_stop_in_factor", C.c_double), ("r_stop_out_factor", C.c_double), ("tau_cutoff", C.c_double),
        ("model", C.c_double * 16),
        ("tp_over_te", C.c_double), ("gamma_ad", C.c_double),
        ("x1_min", C.c_double), ("x1_max", C.c_double), ("t0", C.c_double), ("dt_snap", C.c_double),
        ("freq_hz", C.POINTER(C.c_double)), ("grid_host", C.c_void_p), ("grid_bytes", C.c_uint64),
        ("nx", C.c_int32), ("ny", C.c_int32), ("integrator", C.c_int32), ("step_policy", C.c_int32),
        ("max_steps", C.c_int32), ("n_freq", C.c_int32), ("plasma_model", C.c_int32), ("k2_mode", C.c_int32),
        ("n1", C.c_int32), ("n2", C.c_int32), ("n3", C.c_int32), ("nt", C.c_int32),
        ("grid_dtype", C.c_int32), ("slow_light", C.c_int32), ("snapshot", C.c_int32), ("te_model", C.c_int32),
        ("precision", C.c_int32), ("reserved_", C.c_int32),
    ]


class RaptorError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"raptor error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """The loaded shared library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1801_10452_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, i32, u64p, dp = C.c_void_p, C.c_int32, C.POINTER(C.c_uint64), C.POINTER(C.c_double)
        L.raptor_create.argtypes = [C.POINTER(RaptorParams), C.POINTER(vp)]
        L.raptor_upload_grid.argtypes = [vp, vp, C.c_uint64, vp]
        L.raptor_set_shard.argtypes = [vp, i32, i32]
        L.raptor_render.argtypes = [vp, vp, vp, vp, vp]
        L.raptor_set_camera_time.argtypes = [vp, C.c_double]
        L.raptor_set_window.argtypes = [vp, C.c_int64]
        L.raptor_upload_snapshot.argtypes = [vp, C.c_int64, vp, C.c_uint64, vp]
        L.raptor_light_curve.argtypes = [vp, i32, C.c_double, C.c_double, vp, vp]
        L.raptor_calibrate_delay.argtypes = [i32, vp, vp, i32, vp, vp, C.c_double, i32, dp, dp]
        L.raptor_render_disk.argtypes = [vp, vp, vp, vp, vp, vp]
        L.raptor_line_profile.argtypes = [vp, vp, vp, i32, C.c_double, C.c_double, vp, vp]
        L.raptor_spectrum.argtypes = [vp, vp, vp, vp]
        L.raptor_flux.argtypes = [vp, vp, vp, vp]
        L.raptor_flux_static.argtypes = [vp, C.c_uint64, i32, C.c_double, vp, vp]
        L.raptor_render_host.argtypes = [vp, vp, vp, vp, vp]
        L.raptor_trace.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp]
        L.raptor_eval_rhs.argtypes = [vp, i32, vp, vp, vp]
        L.raptor_null_norm.argtypes = [vp, i32, vp, vp, vp, vp]
        L.raptor_set_null_monitor.argtypes = [vp, vp, C.c_uint64]
        L.raptor_get_counters.argtypes = [vp, u64p, u64p, u64p]
        L.raptor_fp64_peak.argtypes = [i32, dp, dp]
        L.raptor_fp32_peak.argtypes = [i32, dp, dp]
        L.raptor_fp64_probe.argtypes = [i32, i32, dp, dp]
        L.raptor_destroy.argtypes = [vp]
        L.raptor_last_error.argtypes = [vp]
        L.raptor_last_error.restype = C.c_char_p
        for name in SYMBOLS:
            if name != "raptor_last_error":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(rc, ctx=None):
    if rc != 0:
        raise RaptorError(rc, lib().raptor_last_error(ctx).decode())


def params_from_scene(scene):
    """Marshal a scene (duck-typed, see scenes.Scene) into a raptor_params; returns (params, keepalive)."""
    p = RaptorParams()
    p.struct_size = C.sizeof(RaptorParams)
    p.abi_version = ABI_VERSION
    for name in ("a", "mks_h", "mks_r0", "mass", "r_cam", "incl_deg", "fov_M", "t_cam", "M_bh_g", "D_src_cm",
                 "M_unit_g", "step_c", "step_min", "step_max", "eps", "delta", "eps_polar", "r_stop_in_factor",
                 "r_stop_out_factor", "tau_cutoff", "tp_over_te", "gamma_ad", "x1_min", "x1_max", "t0", "dt_snap"):
        setattr(p, name, float(getattr(scene, name)))
    for name in ("nx", "ny", "integrator", "step_policy", "max_steps", "plasma_model", "k2_mode",
                 "n1", "n2", "n3", "nt", "grid_dtype", "slow_light", "snapshot", "te_model"):
        setattr(p, name, int(getattr(scene, name)))
    p.precision = int(getattr(scene, "precision", 0))
    m = list(scene.model) + [0.0] * 16
    p.model = (C.c_double * 16)(*m[:16])
    freq = np.ascontiguousarray(np.asarray(scene.freq_hz, dtype=np.float64))
    p.n_freq = int(freq.size)
    p.freq_hz = freq.ctypes.data_as(C.POINTER(C.c_double))
    keep = [freq]
    grid = getattr(scene, "grid", None)
    if grid is not None:
        g = np.ascontiguousarray(grid, dtype=np.float32 if scene.grid_dtype == 1 else np.float64)
        p.grid_host = g.ctypes.data
        p.grid_bytes = g.nbytes
        keep.append(g)
    return p, keep


# ---- the C ABI, name for name ---------------------------------------------------------------
def raptor_create(params: RaptorParams) -> C.c_void_p:
    ctx = C.c_void_p()
    _check(lib().raptor_create(C.byref(params), C.byref(ctx)))
    return ctx


def raptor_destroy(ctx):
    _check(lib().raptor_destroy(ctx))


def raptor_render(ctx, d_image, d_status=None, d_nsteps=None, stream=None):
    _check(lib().raptor_render(ctx, d_image, d_status, d_nsteps, stream), ctx)


def raptor_render_disk(ctx, d_image, d_redshift, d_status=None, d_nsteps=None, stream=None):
    _check(lib().raptor_render_disk(ctx, d_image, d_redshift, d_status, d_nsteps, stream), ctx)


def raptor_line_profile(ctx, d_image, d_redshift, nbins, g_min, g_max, d_hist, stream=None):
    _check(lib().raptor_line_profile(ctx, d_image, d_redshift, int(nbins), float(g_min), float(g_max), d_hist, stream), ctx)


def raptor_set_camera_time(ctx, t_cam):
    _check(lib().raptor_set_camera_time(ctx, float(t_cam)), ctx)


def raptor_set_window(ctx, first_snapshot):
    _check(lib().raptor_set_window(ctx, int(first_snapshot)), ctx)


def raptor_upload_snapshot(ctx, snapshot, h_snapshot, nbytes, stream=None):
    _check(lib().raptor_upload_snapshot(ctx, int(snapshot), h_snapshot, nbytes, stream), ctx)


def raptor_light_curve(ctx, n_frames, t_cam0, dt_frame, d_flux, stream=None):
    _check(lib().raptor_light_curve(ctx, int(n_frames), float(t_cam0), float(dt_frame), d_flux, stream), ctx)


def raptor_calibrate_delay(t_fast, F_fast, t_slow, F_slow, max_shift, n_grid=2001):
    """Sect. 5.1: (delay, rms) that best aligns the slow-light curve with the fast-light one (raptor.h)."""
    tf, Ff = (np.ascontiguousarray(x, dtype=np.float64) for x in (t_fast, F_fast))
    ts, Fs = (np.ascontiguousarray(x, dtype=np.float64) for x in (t_slow, F_slow))
    d, r = C.c_double(), C.c_double()
    _check(lib().raptor_calibrate_delay(tf.size, tf.ctypes.data, Ff.ctypes.data, ts.size, ts.ctypes.data, Fs.ctypes.data,
                                        float(max_shift), int(n_grid), C.byref(d), C.byref(r)))
    return d.value, r.value


def raptor_set_shard(ctx, rank, world):
    _check(lib().raptor_set_shard(ctx, int(rank), int(world)), ctx)


def raptor_spectrum(ctx, d_flux, d_image=None, stream=None):
    _check(lib().raptor_spectrum(ctx, d_flux, d_image, stream), ctx)


def raptor_flux(ctx, d_image, d_flux, stream=None):
    _check(lib().raptor_flux(ctx, d_image, d_flux, stream), ctx)


def raptor_flux_static(d_image, npix, n_planes, scale, d_flux, stream=None):
    """Flux reduction without a context and without any device allocation (raptor.h): for callers that may not
    call cudaMalloc.  d_image [n_planes][npix] and d_flux [n_planes] are device addresses owned by the caller."""
    _check(lib().raptor_flux_static(d_image, int(npix), int(n_planes), float(scale), d_flux, stream))


def raptor_render_host(ctx, h_image, h_status=None, h_nsteps=None, h_flux=None):
    _check(lib().raptor_render_host(ctx, h_image, h_status, h_nsteps, h_flux), ctx)


def raptor_upload_grid(ctx, h_grid, nbytes, stream=None):
    _check(lib().raptor_upload_grid(ctx, h_grid, nbytes, stream), ctx)


def raptor_trace(ctx, n, d_alpha, d_beta, d_I=None, d_tau=None, d_XK=None, d_status=None, d_nsteps=None, stream=None):
    _check(lib().raptor_trace(ctx, n, d_alpha, d_beta, d_I, d_tau, d_XK, d_status, d_nsteps, stream), ctx)


def raptor_eval_rhs(ctx, n, d_XK, d_f, stream=None):
    _check(lib().raptor_eval_rhs(ctx, n, d_XK, d_f, stream), ctx)


def raptor_null_norm(ctx, n, d_XK, d_out, d_ELQ=None, stream=None):
    _check(lib().raptor_null_norm(ctx, n, d_XK, d_out, d_ELQ, stream), ctx)


def raptor_set_null_monitor(ctx, d_null_max=None, capacity=0):
    """capacity: float64 elements the buffer holds; calls that would write more are refused while it is set (raptor.h)."""
    _check(lib().raptor_set_null_monitor(ctx, d_null_max, int(capacity)), ctx)


def raptor_get_counters(ctx):
    a, b, c = C.c_uint64(), C.c_uint64(), C.c_uint64()
    _check(lib().raptor_get_counters(ctx, C.byref(a), C.byref(b), C.byref(c)), ctx)
    return a.value, b.value, c.value


def raptor_fp64_peak(iters: int = 1 << 16):
    tf, ms = C.c_double(), C.c_double()
    _check(lib().raptor_fp64_peak(int(iters), C.byref(tf), C.byref(ms)))
    return tf.value, ms.value


def raptor_fp32_peak(iters: int = 1 << 16):
    """(TFLOP/s, ms) of independent FFMA chains on all SMs: the measured FP32 peak (raptor.h)."""
    tf, ms = C.c_double(), C.c_double()
    _check(lib().raptor_fp32_peak(int(iters), C.byref(tf), C.byref(ms)))
    return tf.value, ms.value


def raptor_fp64_probe(form: int, iters: int = 1 << 13):
    """(warp instructions per second over the device, nominal SM clock in Hz) for operand form 0..4 (raptor.h)."""
    rate, clk = C.c_double(), C.c_double()
    _check(lib().raptor_fp64_probe(int(form), int(iters), C.byref(rate), C.byref(clk)))
    return rate.value, clk.value


# ---- convenience wrapper ----------------------------------------------------------------------
def _stream_ptr():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Raptor:
    """Context for one scene.  Outputs are torch CUDA tensors allocated here; the kernels fill them."""

    def __init__(self, scene):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1801_10452_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.scene = scene
        self.params, self._keep = params_from_scene(scene)
        self.ctx = raptor_create(self.params)
        self.nf, self.ny, self.nx = self.params.n_freq, self.params.ny, self.params.nx

    def close(self):
        if getattr(self, "ctx", None):
            raptor_destroy(self.ctx)
            self.ctx = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def render(self, want_status=True, image=None):
        import torch
        dev = "cuda"
        if image is None:
            image = torch.empty((self.nf, self.ny, self.nx), dtype=torch.float64, device=dev)
        status = torch.empty((self.ny, self.nx), dtype=torch.int32, device=dev) if want_status else None
        nsteps = torch.empty((self.ny, self.nx), dtype=torch.int32, device=dev) if want_status else None
        raptor_render(self.ctx, image.data_ptr(), status.data_ptr() if want_status else None,
                      nsteps.data_ptr() if want_status else None, _stream_ptr())
        return (image, status, nsteps) if want_status else image

    def render_disk(self):
        """Thin-disk workload: (image [ny][nx], redshift [ny][nx], status, nsteps) as CUDA tensors."""
        import torch
        image = torch.empty((self.ny, self.nx), dtype=torch.float64, device="cuda")
        red = torch.empty((self.ny, self.nx), dtype=torch.float64, device="cuda")
        status = torch.empty((self.ny, self.nx), dtype=torch.int32, device="cuda")
        nsteps = torch.empty((self.ny, self.nx), dtype=torch.int32, device="cuda")
        raptor_render_disk(self.ctx, image.data_ptr(), red.data_ptr(), status.data_ptr(), nsteps.data_ptr(), _stream_ptr())
        return image, red, status, nsteps

    def line_profile(self, image, redshift, nbins, g_min, g_max):
        import torch
        hist = torch.empty((int(nbins),), dtype=torch.float64, device="cuda")
        raptor_line_profile(self.ctx, image.data_ptr(), redshift.data_ptr(), nbins, g_min, g_max, hist.data_ptr(), _stream_ptr())
        return hist

    def light_curve(self, n_frames, t_cam0, dt_frame):
        """Fluxes [n_frames][n_freq] (CUDA tensor, Jy) of frames at camera times t_cam0 + f dt_frame."""
        import torch
        flux = torch.empty((int(n_frames), self.nf), dtype=torch.float64, device="cuda")
        raptor_light_curve(self.ctx, n_frames, t_cam0, dt_frame, flux.data_ptr(), _stream_ptr())
        return flux

    def upload_snapshot(self, index, snapshot):
        g = np.ascontiguousarray(snapshot, dtype=np.float32 if self.scene.grid_dtype == 1 else np.float64)
        raptor_upload_snapshot(self.ctx, index, g.ctypes.data, g.nbytes, None)
        import torch
        torch.cuda.synchronize()

    def set_window(self, first_snapshot):
        raptor_set_window(self.ctx, first_snapshot)

    def set_camera_time(self, t_cam):
        raptor_set_camera_time(self.ctx, t_cam)

    def set_shard(self, rank, world):
        raptor_set_shard(self.ctx, rank, world)

    def flux(self, image):
        import torch
        out = torch.empty((self.nf,), dtype=torch.float64, device="cuda")
        raptor_flux(self.ctx, image.data_ptr(), out.data_ptr(), _stream_ptr())
        return out

    def spectrum(self, image=None):
        import torch
        out = torch.empty((self.nf,), dtype=torch.float64, device="cuda")
        raptor_spectrum(self.ctx, out.data_ptr(), image.data_ptr() if image is not None else None, _stream_ptr())
        return out

    def render_host(self, want_status=False, want_flux=True):
        image = np.empty((self.nf, self.ny, self.nx))
        status = np.empty((self.ny, self.nx), dtype=np.int32) if want_status else None
        nsteps = np.empty((self.ny, self.nx), dtype=np.int32) if want_status else None
        flux = np.empty((self.nf,)) if want_flux else None
        raptor_render_host(self.ctx, image.ctypes.data, status.ctypes.data if want_status else None,
                           nsteps.ctypes.data if want_status else None, flux.ctypes.data if want_flux else None)
        return dict(image=image, status=status, nsteps=nsteps, flux=flux)

    def upload_grid(self, grid):
        g = np.ascontiguousarray(grid, dtype=np.float32 if self.scene.grid_dtype == 1 else np.float64)
        raptor_upload_grid(self.ctx, g.ctypes.data, g.nbytes, _stream_ptr())
        import torch
        torch.cuda.current_stream().synchronize()      # g may be a temporary

    def trace(self, alpha, beta, monitor_null=False):
        import torch
        al = torch.as_tensor(np.asarray(alpha, dtype=np.float64)).cuda()
        be = torch.as_tensor(np.asarray(beta, dtype=np.float64)).cuda()
        n = al.numel()
        I = torch.empty((self.nf, n), dtype=torch.float64, device="cuda")
        tau = torch.empty((self.nf, n), dtype=torch.float64, device="cuda")
        XK = torch.empty((n, 8), dtype=torch.float64, device="cuda")
        status = torch.empty((n,), dtype=torch.int32, device="cuda")
        nsteps = torch.empty((n,), dtype=torch.int32, device="cuda")
        nmax = torch.zeros((n,), dtype=torch.float64, device="cuda") if monitor_null else None
        if monitor_null:
            raptor_set_null_monitor(self.ctx, nmax.data_ptr(), n)
        try:
            raptor_trace(self.ctx, n, al.data_ptr(), be.data_ptr(), I.data_ptr(), tau.data_ptr(), XK.data_ptr(),
                         status.data_ptr(), nsteps.data_ptr(), _stream_ptr())
            torch.cuda.synchronize()
        finally:
            if monitor_null:
                raptor_set_null_monitor(self.ctx, None)
        out = dict(I=I.cpu().numpy(), tau=tau.cpu().numpy(), XK=XK.cpu().numpy(),
                   status=status.cpu().numpy(), nsteps=nsteps.cpu().numpy())
        if monitor_null:
            out["null_max"] = nmax.cpu().numpy()
        return out

    def eval_rhs(self, XK):
        import torch
        q = torch.as_tensor(np.ascontiguousarray(XK, dtype=np.float64)).cuda()
        f = torch.empty((q.shape[0], 4), dtype=torch.float64, device="cuda")
        raptor_eval_rhs(self.ctx, q.shape[0], q.data_ptr(), f.data_ptr(), _stream_ptr())
        torch.cuda.synchronize()
        return f.cpu().numpy()

    def null_norm(self, XK, with_constants=False):
        """g_mn k^m k^n (Eq. 4) at the states XK[n][8]; with_constants: also (E, L, Q) of Eq. 38-40, [n][3]."""
        import torch
        q = torch.as_tensor(np.ascontiguousarray(XK, dtype=np.float64)).cuda()
        out = torch.empty((q.shape[0],), dtype=torch.float64, device="cuda")
        elq = torch.empty((q.shape[0], 3), dtype=torch.float64, device="cuda") if with_constants else None
        raptor_null_norm(self.ctx, q.shape[0], q.data_ptr(), out.data_ptr(), elq.data_ptr() if with_constants else None,
                         _stream_ptr())
        torch.cuda.synchronize()
        return (out.cpu().numpy(), elq.cpu().numpy()) if with_constants else out.cpu().numpy()

    def counters(self):
        return raptor_get_counters(self.ctx)
