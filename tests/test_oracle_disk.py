"""Pins of the oracle's thin-disk workload (Sect. 4.2.1; Fig. 5-6).
None of the expected values comes from the oracle or from the CUDA path:

D1  ISCO radius: 6 M (a = 0), -> 1 M / 9 M (a -> +1 / -1) and the Kerr value for a = 0.9375 (Bardeen et al. 1972)
D2  redshift factor of every crossing equals the closed form for a circular equatorial emitter and a photon with
    conserved E = 1, L = -alpha sin i (Eq. 25): g = 1/(u^t (1 - Omega L)),
    u^t = (r^{3/2} + a)/sqrt(r^3 - 3 r^2 + 2 a r^{3/2}), Omega = 1/(r^{3/2} + a)
D3  flat space (mass 0): the crossing point is where the straight line through the recorded path meets z = 0
D4  face-on Schwarzschild limit: L -> 0, g = sqrt(1 - 3/r): the redshift is a function of the radius alone
D5  image orders: max_order = 1 counts one crossing per ray; higher orders only add intensity; nothing outside
    [r_ISCO, r_out]; the approaching side (alpha < 0 here, L > 0) is blue-shifted relative to the receding one
D6  line profile: sums to the total flux of the counted pixels; support inside the closed-form redshift range
"""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1801_10452_b200 import scenes


def test_D1_isco_radius():
    assert orc.r_isco(0.0) == pytest.approx(6.0, abs=1e-14)
    assert orc.r_isco(1.0 - 1e-12) == pytest.approx(1.0, abs=2e-4)
    assert orc.r_isco(-(1.0 - 1e-12)) == pytest.approx(9.0, abs=1e-6)
    assert orc.r_isco(0.9375) == pytest.approx(2.044201, abs=1e-6)
    # the ISCO is the marginally stable circular orbit: r^2 - 6 r + 8 a sqrt(r) - 3 a^2 = 0 (Bardeen et al. 1972)
    for a in (-0.99, -0.5, 0.3, 0.5, 0.99):
        r = orc.r_isco(a)
        assert r * r - 6 * r + 8 * a * math.sqrt(r) - 3 * a * a == pytest.approx(0.0, abs=1e-12)


def _g_closed(a, r, L):
    ut = (r ** 1.5 + a) / math.sqrt(r ** 3 - 3 * r * r + 2 * a * r ** 1.5)
    Om = 1.0 / (r ** 1.5 + a)
    return 1.0 / (ut * (1.0 - Om * L))


def _crossings(o, al, be):
    """All plane crossings of a ray from its recorded path, found independently of the oracle's detector:
    sign changes of cos(theta) along the path, linear interpolation in the path index."""
    res = o.trace(al, be, record_path=True)
    X0, K0 = o.camera(al, be)
    path = np.vstack([np.concatenate([X0, K0])[None, :], res["path"]])
    th = np.array([orc.mks_theta(o.scene.mks_h, x2)[0] for x2 in path[:, 2]])
    c = np.cos(th)
    out = []
    for i in np.nonzero(c[:-1] * c[1:] < 0)[0]:
        w = c[i] / (c[i] - c[i + 1])
        r = math.exp(path[i, 1] + w * (path[i + 1, 1] - path[i, 1]))
        out.append(r)
    return res, out


@pytest.mark.parametrize("a,incl,h", [(0.0, 60.0, 1.0), (0.9375, 75.0, 1.0), (-0.5, 40.0, 0.3), (0.5, 85.0, 0.3)])
def test_D2_redshift_matches_the_conserved_quantity_closed_form(a, incl, h):
    s = scenes.thin_disk(a=a, incl_deg=incl, max_order=1, mks_h=h)
    o = orc.Oracle(s)
    rng = np.random.default_rng(3)
    n = 0
    for al, be in zip(rng.uniform(-14, 14, 40), rng.uniform(-9, 9, 40)):
        res, rx = _crossings(o, al, be)
        r_in = orc.r_isco(a)
        first_ok = len(rx) > 0 and r_in <= rx[0] <= 15.0
        assert (res["nsampled"] == 1) == first_ok, (al, be, rx)
        if not first_ok:
            assert res["I"][0] == 0.0 and res["tau"][0] == 0.0
            continue
        n += 1
        L = -al * math.sin(math.radians(incl))
        g = res["tau"][0]
        # crossing radius: cos(theta)-linear (here) vs x2-linear (oracle) interpolation differ at O(h^2)
        assert g == pytest.approx(_g_closed(a, rx[0], L), rel=3e-4), (al, be)
        assert res["I"][0] == pytest.approx(g ** 3 / rx[0] ** 2, rel=2e-3)
    assert n >= 8


def test_D3_flat_space_crossing_point():
    s = scenes.thin_disk(a=0.0, incl_deg=50.0, max_order=1, mass=0.0, r_in=0.5, r_out=30.0, r_cam=100.0,
                         step_c=0.01, step_max=0.1)
    o = orc.Oracle(s)
    for al, be in [(3.0, -4.0), (-6.0, 2.0), (0.5, 7.0)]:
        res = o.trace(al, be, record_path=True)
        X0, _ = o.camera(al, be)
        path = np.vstack([np.concatenate([X0, np.zeros(4)])[None, :], res["path"]])
        r, th, ph = np.exp(path[:, 1]), math.pi * path[:, 2], path[:, 3]
        xyz = np.stack([r * np.sin(th) * np.cos(ph), r * np.sin(th) * np.sin(ph), r * np.cos(th)], 1)
        # straight line through the first and last recorded points; where it meets z = 0
        d = xyz[-1] - xyz[0]
        t = -xyz[0, 2] / d[2]
        hit = xyz[0] + t * d
        r_hit = math.hypot(hit[0], hit[1])
        assert res["nsampled"] == 1
        # static emitter limit does not exist for m = 0 (Omega = r^-3/2 is just a rotation speed); use I = g^3/r^2
        # and g from the closed form with u^t = 1/sqrt(1 - r^2 Omega^2) in flat space
        Om = r_hit ** -1.5
        ut = 1.0 / math.sqrt(1.0 - r_hit ** 2 * Om ** 2)
        L = -al * math.sin(math.radians(50.0))
        assert res["tau"][0] == pytest.approx(1.0 / (ut * (1.0 - Om * L)), rel=2e-5)
        assert (res["tau"][0] ** 3 / res["I"][0]) ** 0.5 == pytest.approx(r_hit, rel=2e-5)


def test_D4_face_on_schwarzschild_redshift_depends_on_radius_only():
    s = scenes.thin_disk(a=0.0, incl_deg=0.5, max_order=1)
    o = orc.Oracle(s)
    for al, be in [(7.0, 0.0), (0.0, 9.0), (-8.0, -6.0), (5.0, 11.0)]:
        res, rx = _crossings(o, al, be)
        assert res["nsampled"] == 1
        L = -al * math.sin(math.radians(0.5))
        assert res["tau"][0] == pytest.approx(math.sqrt(1.0 - 3.0 / rx[0]) / (1.0 - L * rx[0] ** -1.5), rel=3e-4)
        assert abs(res["tau"][0] / math.sqrt(1.0 - 3.0 / rx[0]) - 1.0) < 6e-3


def test_D5_orders_support_and_doppler_asymmetry():
    s1 = scenes.thin_disk(a=0.5, incl_deg=70.0, nx=48, max_order=1)
    s10 = replace(s1, model=(0.0, 15.0, 10.0, 3.0) + (0.0,) * 12)
    o1, o10 = orc.Oracle(s1), orc.Oracle(s10)
    r1, r10 = o1.render_disk(), o10.render_disk()
    I1, I10, g1 = r1["image"][0], r10["image"][0], r1["redshift"][0]
    assert np.all(I10 >= I1 - 1e-300) and (I10 > I1 * (1 + 1e-9)).sum() > 10       # lensed images add
    assert ((I1 > 0) == (g1 > 0)).all() and (I1 > 0).sum() > 200
    # I = g^3 / r^2 with r_isco <= r <= 15: bounds on I / g^3
    q = I1[I1 > 0] / g1[I1 > 0] ** 3
    assert q.min() >= 1 / 15.0 ** 2 * (1 - 1e-9) and q.max() <= 1 / orc.r_isco(0.5) ** 2 * (1 + 1e-9)
    # approaching side: L > 0 <=> alpha < 0 (Eq. 25) -> left half of the image is bluer
    left, right = g1[:, :24], g1[:, 24:]
    assert left[left > 0].mean() > right[right > 0].mean() + 0.1
    assert g1.max() > 1.0 and g1[g1 > 0].min() < 0.7


def test_D6_line_profile_sums_to_the_flux_and_stays_in_the_closed_form_range():
    s = scenes.thin_disk(a=0.5, incl_deg=70.0, nx=48, max_order=1)
    o = orc.Oracle(s)
    r = o.render_disk()
    hist = o.line_profile(r["image"], r["redshift"], 60, 0.0, 1.5)
    area = (s.fov_M / s.nx) ** 2
    assert hist.sum() == pytest.approx(r["image"].sum() * area, rel=1e-12)
    # extreme redshift factors of the disk: |L| <= b_max sin i with the photon's impact parameter bounded by the
    # image half-diagonal; scan the closed form over r in [r_isco, 15] and L/E in [-20, 20] sin i for the range
    rr = np.linspace(orc.r_isco(0.5), 15.0, 400)
    Lm = 20.0 * math.sin(math.radians(70.0))
    gmax = max(_g_closed(0.5, x, min(Lm, 0.999 * (x ** 1.5 + 0.5))) for x in rr if True)
    edges = np.linspace(0.0, 1.5, 61)
    nz = np.nonzero(hist)[0]
    assert edges[nz[-1]] < min(gmax, 1.5) and edges[nz[0] + 1] > 0.05
    # numpy's histogram of the same image (same binning rule) is identical
    g, I = r["redshift"].ravel(), r["image"].ravel()
    m = g > 0
    ref = np.histogram(g[m], bins=60, range=(0.0, 1.5), weights=I[m] * area)[0]
    assert np.allclose(hist, ref, rtol=1e-12, atol=0)
