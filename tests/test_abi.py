"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol include/raptor.h
declares, the ctypes struct matches the C struct, and parameter validation (which runs before any CUDA
call) rejects bad input with a message.  No compute call is made here."""
import ctypes as C
import math
import os
import re
from dataclasses import replace

import pytest

from paper_1801_10452_b200 import binding, build, scenes

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def test_library_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "raptor.h")).read()
    declared = set(re.findall(r"\b(raptor_[a-z0-9_]+)\s*\(", header))
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_layout_matches_the_header(lib):
    # struct_size is checked by raptor_create before anything else: a wrong size is EINVAL naming both sizes
    p, keep = binding.params_from_scene(scenes.config_C0(8))
    p.struct_size = 8
    ctx = C.c_void_p()
    rc = lib.raptor_create(C.byref(p), C.byref(ctx))
    assert rc == binding.EINVAL and not ctx.value
    msg = lib.raptor_last_error(None).decode()
    assert "struct_size" in msg and str(C.sizeof(binding.RaptorParams)) in msg


@pytest.mark.parametrize("field,value,needle", [
    ("a", 1.0, "spin"), ("a", float("nan"), "spin"), ("incl_deg", 0.0, "inclination"), ("incl_deg", 180.0, "inclination"),
    ("nx", 0, "nx"), ("r_cam", 1.5, "r_cam"), ("mks_h", 0.0, "mks_h"), ("max_steps", 0, "max_steps"),
    ("integrator", 4, "integrator"), ("k2_mode", 2, "k2_mode"), ("plasma_model", 9, "plasma_model"),
    ("step_min", 0.0, "policy A"), ("fov_M", -1.0, "fov_M"), ("tau_cutoff", float("nan"), "tau_cutoff"),
])
def test_validation_rejects_bad_parameters(lib, field, value, needle):
    s = replace(scenes.config_C0(8), **{field: value})
    p, keep = binding.params_from_scene(s)
    ctx = C.c_void_p()
    rc = lib.raptor_create(C.byref(p), C.byref(ctx))
    assert rc in (binding.EINVAL, binding.EUNSUPPORTED) and not ctx.value
    assert needle in lib.raptor_last_error(None).decode()


def test_validation_of_grid_and_frequencies(lib):
    s = scenes.config_C2(nx=8, n1=16, n2=16)
    p, keep = binding.params_from_scene(s)
    p.grid_bytes = p.grid_bytes - 8
    ctx = C.c_void_p()
    assert lib.raptor_create(C.byref(p), C.byref(ctx)) == binding.EINVAL
    assert "grid_bytes" in lib.raptor_last_error(None).decode()
    p, keep = binding.params_from_scene(replace(s, freq_hz=tuple([1e9] * 65)))
    assert lib.raptor_create(C.byref(p), C.byref(ctx)) == binding.EINVAL
    p, keep = binding.params_from_scene(replace(s, freq_hz=(-1.0,)))
    assert lib.raptor_create(C.byref(p), C.byref(ctx)) == binding.EINVAL


def test_null_handles_are_errors_not_crashes(lib):
    assert lib.raptor_render(None, None, None, None, None) == binding.EINVAL
    assert lib.raptor_spectrum(None, None, None, None) == binding.EINVAL
    assert lib.raptor_null_norm(None, 1, None, None, None, None) == binding.EINVAL
    assert lib.raptor_render_disk(None, None, None, None, None, None) == binding.EINVAL
    assert lib.raptor_line_profile(None, None, None, 10, 0.0, 1.0, None, None) == binding.EINVAL
    assert lib.raptor_light_curve(None, 1, 0.0, 1.0, None, None) == binding.EINVAL
    assert lib.raptor_set_window(None, 0) == binding.EINVAL and lib.raptor_set_camera_time(None, 0.0) == binding.EINVAL
    assert lib.raptor_upload_snapshot(None, 0, None, 0, None) == binding.EINVAL
    assert lib.raptor_destroy(None) == binding.OK
    assert isinstance(lib.raptor_last_error(None), bytes)


def test_product_path_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.Raptor(scenes.config_C0(8))


def test_scene_marshalling_round_trip():
    s = scenes.config_C3(nx=12, n_freq=5, n1=16, n2=16)
    p, keep = binding.params_from_scene(s)
    assert p.n_freq == 5 and p.nx == 12 and p.plasma_model == scenes.GRID2D
    assert p.grid_bytes == 16 * 16 * 8 * 8 and math.isinf(p.tau_cutoff)
    assert [p.freq_hz[i] for i in range(5)] == list(s.freq_hz)
