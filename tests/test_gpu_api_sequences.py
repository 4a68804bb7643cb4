"""GPU tests of C-ABI call SEQUENCES on one context, of memory ownership and of the ordering rule of
include/raptor.h.  compute-sanitizer is closed on this GPU pool, so sequences that would expose a dangling
pointer, a double free, a stale scratch buffer or a missing stream dependency are exercised here explicitly."""
import ctypes as C
import math
from dataclasses import replace

import numpy as np
import pytest

from paper_1801_10452_b200 import scenes

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def rb():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1801_10452_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def orc():
    from oracle import oracle
    return oracle


def test_light_curve_line_profile_light_curve_spectrum_on_one_context(rb):
    # raptor_line_profile used to free the light-curve partial buffer (round-1 bug): the second light curve then wrote
    # through a dangling pointer and raptor_destroy freed it twice.  Same context, growing nbins, interleaved calls.
    s = replace(scenes.config_C4(nx=24, n1=32, n2=24, n3=16, nt=8), freq_hz=(86e9, 230e9))
    t0 = s.t_cam - 10.0
    with rb.Raptor(s) as R:
        lc0 = R.light_curve(4, t0, 5.0).cpu().numpy()
        image, status, nsteps = R.render()
        red = torch.rand((s.ny, s.nx), dtype=torch.float64, device="cuda") * 1.5 + 0.01
        hists = []
        for nbins in (8, 64, 16, 512):
            h = R.line_profile(image[0], red, nbins, 0.0, 1.6).cpu().numpy()
            hists.append(h)
            lc = R.light_curve(4, t0, 5.0).cpu().numpy()
            assert np.array_equal(lc, lc0), nbins                # bit-reproducible, buffer intact
        spec = R.spectrum().cpu().numpy()
        flux = R.flux(image).cpu().numpy()
        lc1 = R.light_curve(6, t0, 5.0).cpu().numpy()            # more frames: the partial buffer grows
        assert np.array_equal(lc1[:4], lc0)
        h2 = R.line_profile(image[0], red, 8, 0.0, 1.6).cpu().numpy()
        torch.cuda.synchronize()
    assert np.array_equal(spec, flux) and np.array_equal(h2, hists[0])
    area = (s.fov_M / s.nx) * (s.fov_M / s.ny)
    for h in hists:                                              # every pixel with 0 < g < 1.6 lands in exactly one bin
        assert h.sum() == pytest.approx(float(image[0].sum()) * area, rel=1e-12)
    # frame f of the curve is the flux of an image rendered at that camera time
    with rb.Raptor(replace(s, t_cam=t0 + 2 * 5.0)) as R2:
        assert np.allclose(R2.spectrum().cpu().numpy(), lc0[2], rtol=1e-13, atol=0)


def test_create_destroy_does_not_leak_device_memory(rb):
    s = scenes.config_C2(nx=16, n1=64, n2=64)
    p, keep = rb.params_from_scene(s)

    def cycle(n):
        for _ in range(n):
            ctx = rb.raptor_create(p)
            img = torch.empty((1, 16, 16), dtype=torch.float64, device="cuda")
            flux = torch.empty((1,), dtype=torch.float64, device="cuda")
            rb.raptor_spectrum(ctx, flux.data_ptr(), None, None)        # allocates the scratch image
            host = np.empty((1, 16, 16))                                # kept alive until the call has returned
            rb.raptor_render_host(ctx, host.ctypes.data, None, None, None)
            rb.raptor_destroy(ctx)

    cycle(3)                                                     # warm up allocator pools (cudaMallocAsync, torch)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()                          # cudaMemGetInfo: the whole device, not torch's pool
    cycle(50)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    # one context holds > 0.5 MiB (grid + partials + scratch): 50 leaked contexts would be > 25 MiB
    assert free0 - free1 < 8 * 1024 * 1024, (free0, free1)


def test_shards_through_the_library_owned_image_paths(rb):
    # raptor_spectrum (NULL image) and raptor_render_host render into the context's scratch image: under a shard the
    # tiles of the other ranks must read as zero, not as whatever the scratch held before
    s = replace(scenes.config_C3(nx=44, n_freq=3), ny=26)
    world = 3
    with rb.Raptor(s) as R:
        full_host = R.render_host(want_status=True)              # fills the scratch with the FULL image first
        full_flux = R.spectrum().cpu().numpy()
        acc_img = np.zeros_like(full_host["image"])
        acc_flux = np.zeros_like(full_flux)
        acc_steps = np.zeros_like(full_host["nsteps"])
        for r in range(world):
            R.set_shard(r, world)
            part = R.render_host(want_status=True)
            f_scratch = R.spectrum().cpu().numpy()
            assert np.array_equal(part["flux"], f_scratch)       # both library-owned paths agree
            acc_img += part["image"]
            acc_flux += part["flux"]
            acc_steps += part["nsteps"]
            assert (part["image"] == 0).mean() > 0.5             # two thirds of the pixels belong to other ranks
        R.set_shard(0, 1)
    assert np.array_equal(acc_img, full_host["image"])           # disjoint support: exact
    assert np.array_equal(acc_steps, full_host["nsteps"])
    assert np.allclose(acc_flux, full_flux, rtol=1e-13, atol=0)  # same pixels, different summation order


def test_render_host_orders_itself_after_an_upload_on_another_stream(rb):
    # bench.py's end-to-end leg: an asynchronous host->device grid copy (pinned memory) on one stream, then the
    # host-buffer render on the context's own stream with no synchronisation in between
    s = scenes.config_C2(nx=32)
    g_new = np.ascontiguousarray(s.grid * np.array([1.7, 1.7, 1, 1, 1, 1, 1, 1]))
    with rb.Raptor(replace(s, grid=g_new)) as R:
        want = R.render_host()["image"]
    pinned = torch.from_numpy(g_new.reshape(-1).copy()).pin_memory()
    side = torch.cuda.Stream()
    for _ in range(5):
        with rb.Raptor(s) as R:
            old = R.render_host()["image"]
            rb.raptor_upload_grid(R.ctx, pinned.data_ptr(), pinned.numel() * 8, C.c_void_p(side.cuda_stream))
            got = R.render_host()["image"]
            assert np.array_equal(got, want) and not np.array_equal(old, want)


@pytest.mark.parametrize("x", [600.0, 690.0, 700.0, 705.0, 709.6, 709.78, 709.79, 712.0, 720.0])
def test_wien_tail_corner_of_the_planck_function(rb, orc, x):
    # Eq. 45 at h nu / k T = x around the overflow of exp(x) - 1 (x = 709.78): below it the slab is
    # thick and I = B_nu ~ 1e-260 ... 1e-308; above it B_nu underflows to 0 and there is no absorption [A13].
    # The CUDA path's exp(x) - 1 must stay finite exactly where libm's does.  (Contrived numbers -- a field of
    # 1e19 G keeps the emissivity non-zero in a plasma this cold -- but every branch is reachable through the ABI.)
    H_, ME_, C_ = 6.62607015e-27, 9.1093837e-28, 2.99792458e10
    nu = 1e16
    theta_e = H_ * nu / (x * ME_ * C_ ** 2)
    s = scenes.slab_scene(1e-270, theta_e, 1e19, 8.0, step_c=0.0, step_min=0.25, step_max=0.25, eps_polar=1e30,
                          r_cam=60.0, incl_deg=30.0, nu_hz=nu)
    with rb.Raptor(s) as R:
        g = R.trace([4.0, -2.0], [3.0, 1.0])
    o = orc.Oracle(s)
    for i, (al, be) in enumerate([(4.0, 3.0), (-2.0, 1.0)]):
        r = o.trace(al, be)
        assert r["I"][0] > 0 and np.isfinite(g["I"][0, i]) and np.isfinite(g["tau"][0, i])
        if x >= 690.0:
            assert (r["tau"][0] > 1.0) == (x < 709.785)          # thick below the overflow, no absorption above
        assert g["I"][0, i] == pytest.approx(r["I"][0], rel=1e-10)
        assert g["tau"][0, i] == pytest.approx(r["tau"][0], rel=1e-10, abs=0.0)
