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


def test_null_monitor_buffer_cannot_be_overrun_by_a_larger_call(rb):
    # the monitor pointer stays set across calls; a buffer sized for a 50-ray trace must not receive a 24 x 24 image
    s = scenes.config_C1(24)
    with rb.Raptor(s) as R:
        small = torch.full((50 + 8,), -1.0, dtype=torch.float64, device="cuda")
        rb.raptor_set_null_monitor(R.ctx, small.data_ptr(), 50)
        al = torch.linspace(-9.0, 9.0, 50, dtype=torch.float64, device="cuda")
        be = torch.full((50,), 0.7, dtype=torch.float64, device="cuda")
        rb.raptor_trace(R.ctx, 50, al.data_ptr(), be.data_ptr())              # fits
        with pytest.raises(rb.RaptorError) as err:
            R.render()                                                         # 576 pixels into 50 elements: refused
        assert err.value.code == rb.EINVAL and "null monitor" in str(err.value)
        with pytest.raises(rb.RaptorError):
            rb.raptor_trace(R.ctx, 51, al.data_ptr(), be.data_ptr())
        with pytest.raises(rb.RaptorError):
            R.spectrum()                                                       # goes through raptor_render
        with pytest.raises(rb.RaptorError):
            rb.raptor_set_null_monitor(R.ctx, small.data_ptr(), 0)
        torch.cuda.synchronize()
        got = small.cpu().numpy()
        assert np.all(got[:50] >= 0.0) and np.all(got[50:] == -1.0)           # the trace wrote its 50, nothing went past
        rb.raptor_set_null_monitor(R.ctx, None)
        img0 = R.render(want_status=False)
        big = torch.zeros((s.ny * s.nx,), dtype=torch.float64, device="cuda")
        rb.raptor_set_null_monitor(R.ctx, big.data_ptr(), big.numel())
        img1 = R.render(want_status=False)
        rb.raptor_set_null_monitor(R.ctx, None)
        torch.cuda.synchronize()
        assert float(big.max()) > 0.0 and np.allclose(img1.cpu().numpy(), img0.cpu().numpy(), rtol=1e-9, atol=0)


def test_counters_wait_for_the_context_only_and_shard_is_committed_after_its_table(rb):
    s = scenes.config_C0(32)
    with rb.Raptor(s) as R:
        R.render(want_status=False)
        steps, sampled, rays = R.counters()                                    # no torch synchronize before: the call waits
        assert rays == 32 * 32 and steps > 100 * rays and 0 < sampled <= steps
        with pytest.raises(rb.RaptorError):
            R.set_shard(3, 2)                                                  # refused: previous shard (0, 1) stays
        full = R.render(want_status=False).cpu().numpy()
        R.set_shard(1, 2)
        part = R.render(want_status=False, image=torch.zeros((1, 32, 32), dtype=torch.float64, device="cuda")).cpu().numpy()
        R.set_shard(0, 1)
        torch.cuda.synchronize()
        owned = part != 0.0
        assert 0 < owned.sum() < owned.size and np.array_equal(part[owned], full[owned])
        assert R.counters()[2] == 32 * 32 * 2 + 16 * 32          # rank 1 of 2 owns 16 of the 32 8x4-pixel tiles


def test_grid_cells_with_denormal_huge_or_infinite_values_hold_no_plasma(rb):
    # user-supplied grid data reaches the one-step reciprocals of the sampler, which want positive normal arguments;
    # cells outside (1e-300, 1e300) in density, or with an infinite velocity, are treated as empty instead of
    # poisoning the ray with NaN (compute-sanitizer is closed on this pool, the oracle divides in IEEE: no parity here)
    clean = scenes.config_C2(nx=48, n1=32, n2=32)
    g = np.array(clean.grid, dtype=np.float64, copy=True).reshape(32, 32, 8)
    g[6:12, 10:16, 0] = 4e-310            # denormal density
    g[14:20, 12:18, 0] = 1e305            # density beyond the range
    g[20:25, 14:20, 2] = np.inf           # infinite radial velocity
    g[8:12, 20:24, 0] = 0.0               # empty cells were always allowed
    with rb.Raptor(clean) as R:
        ref, st0, _ = R.render()
        ref = ref.cpu().numpy()
        R.upload_grid(g.reshape(clean.grid.shape))
        img, st1, _ = R.render()
        img, st1 = img.cpu().numpy(), st1.cpu().numpy()
    assert np.all(np.isfinite(img)) and np.all(img >= 0.0)
    assert not np.any(st1 == 5)                                   # RAPTOR_NONFINITE
    changed = img != ref
    assert 0 < changed.sum() < changed.size                        # the patched cells matter to some rays, not to all
    s32 = scenes.config_PB1_f32(nx=48, n1=32, n2=32)
    with rb.Raptor(s32) as R:
        R.upload_grid(g.reshape(s32.grid.shape))
        img32 = R.render(want_status=False).cpu().numpy()
    assert np.all(np.isfinite(img32))
