"""The single-precision build of the oracle (the SAME source, real = float, Table B.1 of the paper
"Single precision: yes") pinned (i) against closed forms at float tolerances and (ii) against the
double build, which tests/test_oracle_*.py pin function by function.  No GPU."""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1801_10452_b200 import scenes

C_, ME_, KB_, H_ = 2.99792458e10, 9.1093837e-28, 1.380649e-16, 6.62607015e-27
F32 = "f32"


def vac(**kw):
    base = dict(a=0.9375, mks_h=0.3, plasma_model=scenes.VACUUM)
    base.update(kw)
    return scenes.Scene(**base)


def test_f32_build_is_single_precision_throughout():
    T = orc.types(F32)
    assert T.REAL is orc.C.c_float and orc.C.sizeof(T.RayResult) == 16 + 4 * 9
    o = orc.Oracle(scenes.config_C1(4), dtype=F32)
    out = o.render()
    assert out["image"].dtype == np.float32
    # a quantity that needs more than 24 bits: 1 + 2^-30 is not representable -> the float build rounds it away
    assert orc.mks_theta(1.0, 1.0 + 2.0 ** -30, dtype=F32)[0] == np.float32(math.pi)
    assert orc.mks_theta(1.0, 1.0 + 2.0 ** -30)[0] != math.pi


def test_f32_metric_camera_and_constants_of_motion():
    for a, incl, h in [(0.9375, 60.0, 0.3), (0.5, 90.0, 1.0)]:
        o = orc.Oracle(vac(a=a, mks_h=h, incl_deg=incl), dtype=F32)
        X = [0.0, 1.7, 0.31, 0.4]
        assert np.allclose(o.metric(X) @ o.metric_inv(X), np.eye(4), atol=2e-5)              # g g^-1 = 1
        for al, be in [(3.0, 4.0), (-7.5, 0.3)]:
            Xc, Kc = o.camera(al, be)
            E, L, Q = o.conserved(Xc, Kc)
            i = math.radians(incl)
            assert E == pytest.approx(1.0, abs=2e-5)                                          # Eq. 25-29 with E = 1
            assert L == pytest.approx(-al * math.sin(i), abs=2e-3)                            # k_phi ~ 1e3 x 1e-6 rounding at r = 1000
            assert Q == pytest.approx(be ** 2 + math.cos(i) ** 2 * (al ** 2 - a * a), rel=2e-3, abs=5e-2)
            assert abs(o.null_norm(Xc, Kc)) < 1e-4                                            # Eq. 4 (k^t ~ 1)


def test_f32_step_rules_by_hand():
    o = orc.Oracle(vac(step_policy=1, eps=0.03, delta=1e-40), dtype=F32)
    K = [7.7, 0.5, -0.25, 0.1]
    assert o.step_size([0.0, 2.0, 0.2, 1.0], K) == pytest.approx(0.03 / 1.85, rel=1e-6)       # Eq. 21-24
    assert o.step_size([0.0, 2.0, 1.3, 1.0], K) == pytest.approx(0.03 / (0.5 + 0.25 / 0.3 + 0.1), rel=2e-6)
    oA = orc.Oracle(vac(mks_h=1.0), dtype=F32)
    rH = 1.0 + math.sqrt(1.0 - 0.9375 ** 2)
    assert oA.step_size([0, math.log(3.0), 0.5, 0], K) == pytest.approx(0.05 * (3.0 - rH), rel=1e-5)


def test_f32_transfer_closed_forms():
    # Eq. 35: uniform medium, unequal steps: I = S (1 - exp(-tau))
    rng = np.random.default_rng(7)
    j, alpha, nu_hat, Lcm = 3e-18, 2e-13, 1.7, 6.6e11
    I, tau, length = 0.0, 0.0, 0.0
    for h in rng.uniform(0.01, 2.0, size=40):
        I, tau = orc.transfer_update(I, tau, j, alpha, nu_hat, Lcm, float(h), dtype=F32)
        length += float(h)
    assert tau == pytest.approx(nu_hat * alpha * Lcm * length, rel=1e-5)
    assert I == pytest.approx(j / alpha / nu_hat ** 3 * (1 - math.exp(-nu_hat * alpha * Lcm * length)), rel=2e-5)
    # Eq. 45 and the Rayleigh-Jeans limit
    T = 10.0 * ME_ * C_ ** 2 / KB_
    assert orc.planck(230e9, 10.0, dtype=F32) == pytest.approx(2 * H_ * 230e9 ** 3 / C_ ** 2 / math.expm1(H_ * 230e9 / (KB_ * T)), rel=1e-5)
    # Eq. 42-44: same scaling law as the double build, and the same value to float accuracy
    j1, j2 = orc.emissivity(1e11, 1.0, 3.0, 10.0, 0.5, dtype=F32), orc.emissivity(2e11, 1.0, 3.0, 20.0, 0.5, dtype=F32)
    assert j2 / j1 == pytest.approx(2.0, rel=1e-5)
    assert j1 == pytest.approx(orc.emissivity(1e11, 1.0, 3.0, 10.0, 0.5), rel=2e-5)
    # optically thick slab in flat space: I -> B_nu (P8), thin slab: I = j L
    for n_e, thick in ((1e9, True), (1e-5, False)):
        s = scenes.slab_scene(n_e, 10.0, 30.0, 8.0, step_c=0.0, step_min=0.05, step_max=0.05, eps_polar=1e30, r_cam=60.0, incl_deg=30.0)
        r32, r64 = orc.Oracle(s, dtype=F32).trace(4.0, 3.0), orc.Oracle(s).trace(4.0, 3.0)
        if thick:
            assert r32["tau"][0] > 100 and r32["I"][0] == pytest.approx(orc.planck(230e9, 10.0), rel=1e-5)
        else:
            # the number of steps inside the slab may differ by one (the face is crossed at float accuracy)
            assert abs(r32["nsampled"] - r64["nsampled"]) <= 1
            assert r32["I"][0] / r32["nsampled"] == pytest.approx(r64["I"][0] / r64["nsampled"], rel=1e-5)


def test_f32_right_hand_side_and_integrators_against_the_double_build():
    s = vac()
    o32, o64 = orc.Oracle(s, dtype=F32), orc.Oracle(s)
    rng = np.random.default_rng(3)
    for _ in range(30):
        X = [0.0, rng.uniform(0.6, 5.0), rng.uniform(0.1, 0.9), 1.0]
        K = list(rng.normal(size=4))
        f32_, f64_ = o32.rhs(X, K), o64.rhs(X, K)
        assert np.abs(f32_ - f64_).max() <= 3e-4 * np.abs(f64_).max()          # Eq. 2 with float metric derivatives
        for step in ("rk4_step", "rk2_step", "verlet_step"):
            X32, K32 = getattr(o32, step)(X, K, -0.01)
            X64, K64 = getattr(o64, step)(X, K, -0.01)
            assert np.abs(X32 - X64).max() <= 2e-6 * max(1.0, np.abs(X64).max()) and np.abs(K32 - K64).max() <= 1e-5 * np.abs(K64).max()
    # flat space: straight lines at float accuracy (P7)
    o = orc.Oracle(vac(a=0.0, mks_h=1.0, mass=0.0, incl_deg=50.0, r_cam=100.0, step_c=0.005, step_max=0.05, integrator=3), dtype=F32)
    res = o.trace(3.0, -4.0, record_path=True)
    r, th, ph = np.exp(res["path"][:, 1].astype(float)), math.pi * res["path"][:, 2].astype(float), res["path"][:, 3].astype(float)
    P = np.stack([r * np.sin(th) * np.cos(ph), r * np.sin(th) * np.sin(ph), r * np.cos(th)], 1)
    d = P[-1] - P[0]
    n = d / np.linalg.norm(d)
    dev = (P - P[0]) - np.outer((P - P[0]) @ n, n)
    assert res["status"] == 2 and np.abs(dev).max() < 5e-2                      # over a 200 M path


def test_f32_whole_image_of_the_papers_configuration_against_the_double_build():
    # PB1 = Table B.1: RK2, Eq. 21-24 with eps = 0.03, tau cut-off, on the seeded grid.
    # The FP32-vs-FP64 difference of the image is a result in itself: the median pixel
    # differs by < 1e-3, the total flux by < 1e-3.
    s = scenes.config_PB1(nx=24)
    o32, o64 = orc.Oracle(s, dtype=F32), orc.Oracle(s)
    a, b = o64.render(), o32.render()
    assert (a["status"] == b["status"]).mean() > 0.98
    assert (np.abs(a["nsteps"] - b["nsteps"]) <= 2).mean() > 0.95
    e = np.abs(b["image"] - a["image"]) / np.maximum(np.abs(a["image"]), 1e-30 * np.abs(a["image"]).max())
    assert np.median(e) < 1e-3 and np.quantile(e, 0.9) < 1e-2
    assert o32.flux(b["image"])[0] == pytest.approx(o64.flux(a["image"])[0], rel=1e-3)
