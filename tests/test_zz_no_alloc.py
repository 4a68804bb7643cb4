"""raptor_flux_static: the flux reduction for callers that are not allowed to allocate device memory.

Who that is: a plug-in inside a program whose own memory pool already owns the whole GPU, a job whose device-memory
budget was fixed beforehand, a loop that must stay clear of cudaMalloc's device-wide synchronisation, or code that
holds an image on the device but no raptor context (raptor_create allocates).  The entry point keeps its partial sums
in an array built into the library instead, shared by every call on a device and never cleared, so what is checked
here is: (1) it returns what the allocating path (raptor_flux on a context) returns, bit for bit, which is far inside
the 1e-9 the flux parity tests allow; (2) a second call straight after the first, with a smaller image, is not
disturbed by what the first one left in the array; (3) oversized and malformed requests are refused with a message
and nothing is launched.

The file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide other tests), and
it passes alone in a fresh process as well as after the rest of the suite: the first call does the once-per-device
address look-up, whoever makes it.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1801_10452_b200 import binding, scenes

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

FLUX_RTOL = 1e-9      # the bar of the flux parity tests (tests/test_gpu_parity.py); measured here: bit-equal


def _jy_scale(s):
    """The factor raptor_flux applies (include/raptor.h): 1e23 (fov/nx)(fov/ny) L^2/D^2."""
    return 1e23 * (s.fov_M / s.nx) * (s.fov_M / s.ny) * s.L_cm * s.L_cm / (s.D_src_cm * s.D_src_cm)


def _both_paths(scene, image):
    """(flux of the allocating path, flux of the no-allocation entry point) for the same device image."""
    stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    with binding.Raptor(scene) as r:
        ref = r.flux(image)
        torch.cuda.synchronize()
    out = torch.full((scene.n_freq,), float("nan"), dtype=torch.float64, device="cuda")
    binding.raptor_flux_static(image.data_ptr(), scene.nx * scene.ny, scene.n_freq, _jy_scale(scene), out.data_ptr(), stream)
    torch.cuda.synchronize()
    return ref.cpu().numpy(), out.cpu().numpy()


def test_two_calls_in_a_row_match_the_allocating_path():
    # call 1: a rendered image, 3 planes of 200 x 170 = 34000 pixels = two full chunks of 16384 and a ragged third
    big = scenes.config_C0(64).with_pixels(200, 170)
    big.freq_hz = (43e9, 230e9, 690e9)
    with binding.Raptor(big) as r:
        image = r.render(want_status=False)
        torch.cuda.synchronize()
    ref1, got1 = _both_paths(big, image)
    assert np.all(np.isfinite(got1)) and np.all(ref1 > 0)
    np.testing.assert_allclose(got1, ref1, rtol=FLUX_RTOL, atol=0.0)
    assert np.array_equal(got1, ref1)              # same chunks, same tree: not merely close

    # call 2, directly afterwards: fewer planes and fewer chunks, signed values; the array still holds call 1's sums
    small = scenes.config_C0(64).with_pixels(150, 120)
    small.freq_hz = (86e9, 345e9)
    gen = torch.Generator(device="cpu").manual_seed(1801_10452)
    image2 = torch.randn((2, 120, 150), dtype=torch.float64, generator=gen).cuda()
    ref2, got2 = _both_paths(small, image2)
    np.testing.assert_allclose(got2, ref2, rtol=FLUX_RTOL, atol=0.0)
    assert np.array_equal(got2, ref2)
    # and against a sum that neither path computed: float64 pairwise sum on the host (rounding order differs)
    host = image2.cpu().numpy().reshape(2, -1).sum(1) * _jy_scale(small)
    np.testing.assert_allclose(got2, host, rtol=0.0, atol=1e-12 * np.abs(image2.cpu().numpy()).sum() * _jy_scale(small))

    # call 3: the first image again gives the first answer again (nothing of call 2 leaks back)
    _, again = _both_paths(big, image)
    assert np.array_equal(again, got1)


def test_limits_are_refused_with_a_message():
    img = torch.zeros((4,), dtype=torch.float64, device="cuda")
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    limit = 16384                                   # RAPTOR_FLUX_STATIC_MAX_PARTIALS
    cases = [
        (img.data_ptr(), 16384 * limit + 1, 1),     # one chunk too many for a single plane
        (img.data_ptr(), 16384 * 2, limit // 2 + 1),  # planes x chunks over the limit
        (img.data_ptr(), 0, 1), (img.data_ptr(), 4, 0), (None, 4, 1),
    ]
    for ptr, npix, planes in cases:
        with pytest.raises(binding.RaptorError) as err:
            binding.raptor_flux_static(ptr, npix, planes, 1.0, out.data_ptr())
        assert err.value.code == binding.EINVAL and "raptor_flux_static" in str(err.value)
    with pytest.raises(binding.RaptorError):
        binding.raptor_flux_static(img.data_ptr(), 4, 1, 1.0, None)
    torch.cuda.synchronize()
    assert out.item() == 7.0                        # nothing was launched
    # the largest request that fits is accepted as far as the size check goes: 1 plane x 1 chunk here
    binding.raptor_flux_static(img.data_ptr(), 4, 1, 1.0, out.data_ptr())
    torch.cuda.synchronize()
    assert out.item() == 0.0
