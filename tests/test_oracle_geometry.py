"""Pins of the oracle's geometry (metric, connection, camera, stepper) against what GR and the
paper fix -- none of the expected values below comes from the oracle or from the CUDA path.

P1 metric identities + Boyer-Lindquist transform (A.5)
P2 connection: symmetry, textbook components, finite differences of the metric
P3 camera: conserved quantities of Eq. 38-40, Bardeen's critical curve and the
   two 'difficult' orbits of Table 1
P4 null condition Eq. 4
P5 E, L, Q conserved with 4th-order convergence on the Fig. 3 orbit
P6 shadow edge: sqrt(27) M (Schwarzschild) and the Kerr critical curve
P7 flat-space limit: straight lines
P10 chart transforms A.7-A.16
P13 redshift closed forms (Eq. 31)
"""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1801_10452_b200 import scenes

RNG = np.random.default_rng(20180131)


def vac(a=0.0, h=1.0, **kw):
    base = dict(a=a, mks_h=h, plasma_model=scenes.VACUUM)
    base.update(kw)
    return scenes.Scene(**base)


# ------------------------------------------------------------------------- textbook pieces
def g_bl(a, r, th):
    """Boyer-Lindquist Kerr metric, M = 1 (textbook, e.g. Bardeen, Press & Teukolsky 1972)."""
    s2, c2 = math.sin(th) ** 2, math.cos(th) ** 2
    Sig, Del = r * r + a * a * c2, r * r - 2 * r + a * a
    g = np.zeros((4, 4))
    g[0, 0] = -(1 - 2 * r / Sig)
    g[0, 3] = g[3, 0] = -2 * a * r * s2 / Sig
    g[1, 1] = Sig / Del
    g[2, 2] = Sig
    g[3, 3] = ((r * r + a * a) ** 2 - Del * a * a * s2) * s2 / Sig
    return g


def critical_curve(a, r_s):
    """Bardeen (1973) constants of the spherical photon orbit of radius r_s: xi = L/E, eta = Q/E^2."""
    xi = -(r_s ** 3 - 3 * r_s ** 2 + a * a * r_s + a * a) / (a * (r_s - 1))
    eta = r_s ** 3 * (4 * a * a - r_s * (r_s - 3) ** 2) / (a * a * (r_s - 1) ** 2)
    return xi, eta


def photon_orbit_radii(a):
    return (2 * (1 + math.cos(2 / 3 * math.acos(-a))), 2 * (1 + math.cos(2 / 3 * math.acos(a))))  # pro, retro


# ------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("a", [0.0, 0.5, 0.9375, 0.998])
def test_P1_metric_inverse_and_determinant(a):
    for _ in range(20):
        r, th = RNG.uniform(1.1, 60.0), RNG.uniform(0.05, math.pi - 0.05)
        g, gi = orc.metric_ks(a, 1.0, r, th), orc.metric_ks_inv(a, 1.0, r, th)
        assert np.allclose(g, g.T, atol=0)
        assert np.allclose(g @ gi, np.eye(4), atol=1e-12)
        Sig = r * r + (a * math.cos(th)) ** 2
        assert np.linalg.det(g) == pytest.approx(-Sig ** 2 * math.sin(th) ** 2, rel=1e-11)


@pytest.mark.parametrize("a", [0.0, 0.6, 0.9375])
def test_P1_ks_is_the_A5_transform_of_boyer_lindquist(a):
    # k^KS = J k^BL with J the matrix of A.5  =>  g_KS = J^-T g_BL J^-1
    for _ in range(10):
        r, th = RNG.uniform(2.5, 40.0), RNG.uniform(0.1, math.pi - 0.1)
        Del = r * r - 2 * r + a * a
        J = np.eye(4)
        J[0, 1] = 2 * r / Del
        J[3, 1] = a / Del
        Ji = np.linalg.inv(J)
        assert np.allclose(Ji.T @ g_bl(a, r, th) @ Ji, orc.metric_ks(a, 1.0, r, th), rtol=1e-11, atol=1e-11)


@pytest.mark.parametrize("h", [1.0, 0.3])
def test_P1_mks_metric_and_inverse(h):
    o = orc.Oracle(vac(a=0.9375, h=h))
    for _ in range(10):
        X = [0.0, RNG.uniform(0.3, 4.0), RNG.uniform(0.03, 0.97), RNG.uniform(0, 6)]
        g, gi = o.metric(X), o.metric_inv(X)
        assert np.allclose(g @ gi, np.eye(4), atol=1e-11)
        # line element invariance: g_MKS = Lam g_KS Lam with the Jacobian of A.10-A.13
        th, dth, _ = orc.mks_theta(h, X[2])
        r = math.exp(X[1])
        Lam = np.diag([1.0, r, dth, 1.0])
        assert np.allclose(g, Lam @ orc.metric_ks(0.9375, 1.0, r, th) @ Lam, rtol=1e-13)


# ------------------------------------------------------------------------------------- P2
def _fd_dmetric(o, X, c, step=2e-3):
    """Richardson-extrapolated central difference of the oracle's metric along x^c."""
    def D(hh):
        Xp, Xm = list(X), list(X)
        Xp[c] += hh
        Xm[c] -= hh
        return (o.metric(Xp) - o.metric(Xm)) / (2 * hh)
    d1, d2, d4 = D(step), D(step / 2), D(step / 4)
    r1, r2 = (4 * d2 - d1) / 3, (4 * d4 - d2) / 3
    return (16 * r2 - r1) / 15


@pytest.mark.parametrize("a,h", [(0.0, 1.0), (0.9375, 1.0), (0.9375, 0.3), (0.998, 0.3)])
def test_P2_connection_against_finite_differences(a, h):
    o = orc.Oracle(vac(a=a, h=h))
    for _ in range(6):
        X = [0.0, RNG.uniform(0.4, 3.5), RNG.uniform(0.08, 0.92), 1.0]
        dg = np.zeros((4, 4, 4))
        for c in (1, 2):
            dg[c] = _fd_dmetric(o, X, c)
        scale = np.abs(o.metric(X)).max()
        assert np.allclose(o.dmetric(X), dg, atol=2e-9 * scale, rtol=2e-9)
        gi = o.metric_inv(X)
        # Eq. 2 with the finite-difference derivatives
        G = 0.5 * (np.einsum("ar,mnr->amn", gi, dg) + np.einsum("ar,nmr->amn", gi, dg)
                   - np.einsum("ar,rmn->amn", gi, dg))
        Go = o.christoffel(X)
        assert np.allclose(Go, np.swapaxes(Go, 1, 2), atol=1e-13 * np.abs(Go).max())
        assert np.allclose(Go, G, atol=1e-8 * np.abs(Go).max())


def test_P2_textbook_schwarzschild_components():
    # spherical symmetry with areal radius: Gamma^th_{r th} = 1/r, Gamma^ph_{th ph} = cot th,
    # Gamma^th_{ph ph} = -sin th cos th, Gamma^r_{th th} = -(r - 2M) in ingoing Eddington-Finkelstein.
    # In MKS(h=1): x1 = ln r, theta = pi x2.
    o = orc.Oracle(vac(a=0.0, h=1.0))
    for _ in range(5):
        x1, x2 = RNG.uniform(0.8, 3.0), RNG.uniform(0.1, 0.9)
        r, th = math.exp(x1), math.pi * x2
        G = o.christoffel([0, x1, x2, 0])
        assert G[2, 1, 2] == pytest.approx(1.0, rel=1e-12)
        assert G[3, 2, 3] == pytest.approx(math.pi / math.tan(th), rel=1e-12)
        assert G[2, 3, 3] == pytest.approx(-math.sin(th) * math.cos(th) / math.pi, rel=1e-12)
        assert G[3, 1, 3] == pytest.approx(1.0, rel=1e-12)
        assert G[1, 2, 2] == pytest.approx(-(r - 2.0) * math.pi ** 2 / r, rel=1e-12)
        # Gamma^t_tt = 2M^2/r^3 in ingoing EF (t~ = v - r)
        assert G[0, 0, 0] == pytest.approx(2.0 / r ** 3, rel=1e-12)


def test_P2_geodesic_rhs_is_the_contraction_of_eq6():
    o = orc.Oracle(vac(a=0.9375, h=0.3))
    X = [0.0, 1.3, 0.31, 0.4]
    K = [1.3, -0.2, 0.05, 0.07]
    G = o.christoffel(X)
    assert np.allclose(o.rhs(X, K), -np.einsum("amn,m,n->a", G, K, K), rtol=1e-13)


# ------------------------------------------------------------------------------------ P10
@pytest.mark.parametrize("h", [1.0, 0.3, 0.0])
def test_P10_theta_map_derivatives_and_newton_inverse(h):
    for x2 in np.linspace(0.02, 0.98, 25):
        th, d1, d2 = orc.mks_theta(h, x2)
        assert th == pytest.approx(math.pi * x2 + 0.5 * (1 - h) * math.sin(2 * math.pi * x2), abs=1e-15)
        e = 1e-5
        assert d1 == pytest.approx((orc.mks_theta(h, x2 + e)[0] - orc.mks_theta(h, x2 - e)[0]) / (2 * e), rel=1e-7, abs=1e-8)
        assert d2 == pytest.approx((orc.mks_theta(h, x2 + e)[1] - orc.mks_theta(h, x2 - e)[1]) / (2 * e), rel=1e-7, abs=1e-8)
        if h > 0:
            x2_back, iters = orc.x2_of_theta(h, th)
            assert x2_back == pytest.approx(x2, abs=1e-13)
            assert iters < 100


# ------------------------------------------------------------------------------------- P3
@pytest.mark.parametrize("a,incl,h", [(0.9375, 60.0, 1.0), (0.998, 90.0, 0.3), (0.5, 20.0, 0.3)])
def test_P3_camera_reproduces_E_L_Q_of_eq25_26(a, incl, h):
    o = orc.Oracle(vac(a=a, h=h, incl_deg=incl))
    i = math.radians(incl)
    for al, be in [(3.0, 4.0), (-7.5, 0.3), (0.2, -11.0), (-2.1109, 0.0)]:
        X, K = o.camera(al, be)
        E, L, Q = o.conserved(X, K)
        assert E == pytest.approx(1.0, rel=1e-12)
        assert L == pytest.approx(-al * math.sin(i), rel=1e-11, abs=1e-12)                # Eq. 25
        assert Q == pytest.approx(be ** 2 + math.cos(i) ** 2 * (al ** 2 - a * a), rel=1e-9, abs=1e-9)  # Eq. 26 with a^2
        assert abs(o.null_norm(X, K)) < 1e-12                                              # Eq. 4
        assert K[1] > 0 and K[0] > 0                                                       # outgoing, future directed
        assert X[1] == pytest.approx(math.log(o.scene.r_cam)) and X[3] == 0.0
        assert orc.mks_theta(h, X[2])[0] == pytest.approx(i, abs=1e-13)
        # A.6 back to Boyer-Lindquist: lowering with the BL metric must give k_t = -1, k_phi = L
        r, th = o.scene.r_cam, i
        Del = r * r - 2 * r + a * a
        dth = orc.mks_theta(h, X[2])[1]
        k_ks = np.array([K[0], K[1] * r, K[2] * dth, K[3]])
        k_bl = k_ks - np.array([2 * r / Del * k_ks[1], 0, 0, a / Del * k_ks[1]])
        kc = g_bl(a, r, th) @ k_bl
        assert kc[0] == pytest.approx(-1.0, rel=1e-10) and kc[3] == pytest.approx(L, rel=1e-9, abs=1e-10)
        assert kc[2] ** 2 == pytest.approx(be ** 2, rel=1e-9, abs=1e-12)                   # k_theta^2 = beta^2 at the camera


def test_P3_table1_orbits_sit_on_the_critical_curve(golden):
    a = golden["table1_a"]
    r_pro, r_retro = photon_orbit_radii(a)
    xi_pro, _ = critical_curve(a, r_pro)
    # orbit 1: i = 90 deg, beta = 0: L = -alpha sin i must equal the prograde critical xi to the printed digits
    assert -golden["table1_orbit1_alpha"] == pytest.approx(xi_pro, abs=6e-5)
    # orbit 2: i = 60 deg, alpha = -0.001: beta_c = sqrt(eta + a^2 cos^2 i - xi^2 cot^2 i)
    i = math.radians(golden["table1_orbit2_incl"])
    from scipy.optimize import brentq
    xi_target = -golden["table1_orbit2_alpha"] * math.sin(i)
    r_s = brentq(lambda rs: critical_curve(a, rs)[0] - xi_target, r_pro + 1e-9, r_retro - 1e-9)
    xi, eta = critical_curve(a, r_s)
    beta_c = math.sqrt(eta + (a * math.cos(i)) ** 2 - xi ** 2 / math.tan(i) ** 2)
    assert beta_c == pytest.approx(golden["table1_orbit2_beta"], abs=5e-4)


def test_P3_table1_orbit1_winds_around_the_hole(golden):
    # "looping around the horizon many times before plunging in or escaping"
    s = vac(a=golden["table1_a"], h=1.0, incl_deg=golden["table1_orbit1_incl"], r_cam=100.0,
            step_c=0.02, step_max=0.25)
    o = orc.Oracle(s)
    res = o.trace(golden["table1_orbit1_alpha"], golden["table1_orbit1_beta"], record_path=True)
    dphi = abs(res["path"][-1, 3] - res["path"][0, 3])
    assert dphi > 2.5 * 2 * math.pi
    # a ray well outside the critical curve on the same side barely bends
    res2 = o.trace(golden["table1_orbit1_alpha"] - 4.0, 0.0, record_path=True)
    assert abs(res2["path"][-1, 3] - res2["path"][0, 3]) < 1.5 * math.pi and res2["status"] == 2


# ---------------------------------------------------------------------------------- P4, P5
def test_P5_conserved_quantities_converge_at_fourth_order(golden):
    errs = []
    hs = [0.1, 0.05, 0.025]
    for hstep in hs:
        s = vac(a=golden["fig3_a"], h=1.0, incl_deg=golden["fig3_incl"], r_cam=40.0,
                step_c=0.0, step_min=hstep, step_max=hstep, eps_polar=1e30, max_steps=int(round(70.0 / hstep)))
        o = orc.Oracle(s)
        X0, K0 = o.camera(golden["fig3_alpha"], golden["fig3_beta"])
        E0, L0, Q0 = o.conserved(X0, K0)
        res = o.trace(golden["fig3_alpha"], golden["fig3_beta"])
        assert res["status"] == 3 and res["nsteps"] == int(round(70.0 / hstep))   # same affine length every time
        E, L, Q = o.conserved(res["X"], res["K"])
        errs.append([abs(E - E0), abs(L - L0), abs(Q - Q0)])
    errs = np.array(errs)
    slopes = np.log(errs[:-1] / errs[1:]) / np.log(2.0)
    assert np.all(errs[-1] < 1e-8)
    # E and L are in the asymptotic regime; the error of Q changes sign near h = 0.15 (its h^4 and h^5
    # terms compete on this orbit) and approaches the 4th-order line from below
    assert np.all(np.abs(slopes[:, :2] - golden["rk4_order"]) < 0.2), slopes
    assert 3.5 < slopes[-1, 2] < 4.5 and slopes[-1, 2] > slopes[0, 2], slopes


@pytest.mark.parametrize("h", [1.0, 0.3])
def test_P4_P5_null_condition_and_constants_along_a_policy_A_ray(h):
    o = orc.Oracle(vac(a=0.9375, h=h, incl_deg=60.0))
    X0, K0 = o.camera(7.0, 3.0)
    E0, L0, Q0 = o.conserved(X0, K0)
    res = o.trace(7.0, 3.0, monitor_null=True)
    assert res["status"] == 2 and 1500 < res["nsteps"] < 3500
    E, L, Q = o.conserved(res["X"], res["K"])
    assert abs(E - E0) < 1e-4 and abs(L - L0) < 1e-4 and abs(Q - Q0) < 1e-3 * Q0
    assert res["null_max"] < 2e-4      # truncation error of the policy-A steps; |k^t| stays O(1) on this ray


def test_P2_mks_chain_rule_same_ray_in_two_charts():
    # The same geodesic integrated in MKS(h=1) and MKS(h=0.3) differs only by truncation error.
    out = []
    for h in (1.0, 0.3):
        o = orc.Oracle(vac(a=0.9375, h=h, incl_deg=60.0, r_cam=60.0, step_c=0.0, step_min=0.02, step_max=0.02,
                           eps_polar=1e30, max_steps=4000))
        res = o.trace(8.0, 4.0)
        assert res["status"] == 3           # both stop after the same affine length, outside the hole
        th = orc.mks_theta(h, res["X"][2])[0]
        out.append([res["X"][0], res["X"][1], th, res["X"][3]])
    assert np.allclose(out[0], out[1], rtol=0, atol=2e-9)


def test_P2_radial_offset_r0_same_ray_in_two_charts():
    # r = r0 + exp(x1) (A.10): the same geodesic with r0 = 0 and r0 = 0.5 differs only by truncation,
    # and negative spin mirrors the image: (a, alpha) -> (-a, -alpha) flips the sign of phi and leaves r, theta, t
    out = []
    for r0 in (0.0, 0.5):
        o = orc.Oracle(vac(a=0.9375, h=0.3, mks_r0=r0, incl_deg=60.0, r_cam=60.0, step_c=0.0, step_min=0.01,
                           step_max=0.01, eps_polar=1e30, max_steps=8000))
        res = o.trace(8.0, 4.0)
        assert res["status"] == 3
        out.append([res["X"][0], math.log(r0 + math.exp(res["X"][1])), res["X"][2], res["X"][3]])
    assert np.allclose(out[0], out[1], rtol=0, atol=5e-9)
    om = orc.Oracle(vac(a=-0.9375, h=0.3, incl_deg=60.0, r_cam=60.0, step_c=0.0, step_min=0.01, step_max=0.01,
                        eps_polar=1e30, max_steps=8000))
    rm = om.trace(-8.0, 4.0)
    assert np.allclose([rm["X"][0], rm["X"][1], rm["X"][2], -rm["X"][3]],
                       [out[0][0], out[0][1], out[0][2], out[0][3]], rtol=0, atol=1e-11)


# ------------------------------------------------------------------------------------- P6
def _edge(o, direction, lo, hi, tol=2e-6):
    """Bisect along a ray of the image plane for the capture/escape boundary."""
    ux, uy = direction
    assert o.trace(lo * ux, lo * uy)["status"] == 1 and o.trace(hi * ux, hi * uy)["status"] == 2
    while hi - lo > tol:
        mid = 0.5 * (lo + hi)
        if o.trace(mid * ux, mid * uy)["status"] == 1:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def test_P6_schwarzschild_shadow_is_sqrt27():
    o = orc.Oracle(vac(a=0.0, h=1.0, incl_deg=60.0, r_cam=1000.0))
    for ang in (0.3, 2.0):
        b = _edge(o, (math.cos(ang), math.sin(ang)), 4.0, 7.0)
        # the camera sits at r = 1000 M, not at infinity: b_c = sqrt(27) holds for L/E, which Eq. 25-26 fix exactly
        assert b == pytest.approx(math.sqrt(27.0), abs=1e-4)


def test_P6_kerr_shadow_edge_on_the_equator_matches_bardeen():
    a = 0.9375
    o = orc.Oracle(vac(a=a, h=1.0, incl_deg=90.0, r_cam=1000.0))
    r_pro, r_retro = photon_orbit_radii(a)
    xi_pro, xi_retro = critical_curve(a, r_pro)[0], critical_curve(a, r_retro)[0]
    # L = -alpha sin i: prograde edge at alpha = -xi_pro, retrograde at alpha = -xi_retro > 0
    # (beta -> 0+: the exact equator beta = 0 has sign(beta) = 0 and stays in the plane as well)
    e_pro = _edge(o, (-1.0, 1e-9), 1.0, 4.0)
    e_retro = _edge(o, (1.0, 1e-9), 5.0, 9.0)
    assert e_pro == pytest.approx(xi_pro, abs=1e-4)
    assert e_retro == pytest.approx(-xi_retro, abs=1e-4)


# ------------------------------------------------------------------------------------- P7
def _cartesian(a, path):
    r, th, ph = np.exp(path[:, 1]), math.pi * path[:, 2], path[:, 3]
    s = np.sin(th)
    # x + i y = (r + i a) sin(theta) exp(i phi~)  (flat space in the m = 0 Kerr-Schild spheroidal chart)
    return np.stack([s * (r * np.cos(ph) - a * np.sin(ph)), s * (r * np.sin(ph) + a * np.cos(ph)), r * np.cos(th)], 1)


def _line_deviation(a, sc, sm, al=3.0, be=-4.0):
    o = orc.Oracle(vac(a=a, h=1.0, mass=0.0, incl_deg=50.0, r_cam=100.0, step_c=sc, step_max=sm))
    res = o.trace(al, be, record_path=True)
    assert res["status"] == 2
    P = _cartesian(a, res["path"])
    d = P[-1] - P[0]
    n = d / np.linalg.norm(d)
    dev = (P - P[0]) - np.outer((P - P[0]) @ n, n)
    t = res["path"][:, 0]
    closest = P[0] - (P[0] @ n) * n
    return np.abs(dev).max(), abs(t[0] - t[-1]) / np.linalg.norm(d) - 1.0, np.linalg.norm(closest)


@pytest.mark.parametrize("a", [0.0, 0.6])
def test_P7_flat_space_rays_are_straight_lines(a):
    # mass parameter 0: every ray is a straight line of the Cartesian frame, traversed at unit
    # coordinate speed (E = 1); the integrator approaches it at 4th order in the step
    dev_c, dt_c, _ = _line_deviation(a, 0.025, 0.25)
    dev_f, dt_f, closest = _line_deviation(a, 0.005, 0.05)
    assert dev_f < 2e-8 and abs(dt_f) < 1e-10
    assert 5.0 ** 4 / 2 < dev_c / dev_f < 5.0 ** 4 * 2
    if a == 0.0:
        # closest approach to the origin = impact parameter sqrt(alpha^2 + beta^2)
        assert closest == pytest.approx(5.0, abs=2e-8)


# ------------------------------------------------------------------------------------ P13
def test_P13_redshift_of_a_free_falling_emitter_on_a_radial_ray():
    # alpha = beta = 0, a = 0: radial ray.  nu_hat = -k.u = 1/(1 - sqrt(2/r)) for free fall from rest at
    # infinity and an E = 1 outgoing photon (Eq. 31)
    s = replace(scenes.config_C0(8), r_cam=200.0)
    o = orc.Oracle(s)
    res = o.trace(0.0, 0.0, record_path=True)
    for row in res["path"][::150]:
        X, K = row[:4], row[4:]
        r = math.exp(X[1])
        pl = o.plasma(X)
        g = o.metric(X)
        assert pl["u"] @ g @ pl["u"] == pytest.approx(-1.0, rel=1e-12)
        assert pl["u"][1] * r == pytest.approx(-math.sqrt(2.0 / r), rel=1e-12)        # u^r = -sqrt(2M/r)
        nu_hat = -(K @ g @ pl["u"])
        # K carries the truncation error of the policy-A steps, amplified ~1/(r - 2) near the horizon
        assert nu_hat == pytest.approx(1.0 / (1.0 - math.sqrt(2.0 / r)), rel=2e-7 if r > 3.0 else 5e-6)


# ------------------------------------------------------------------------- step rules, pixel grid, layout
# Hand-computed expectations: none of the numbers below comes from orc_step_size / orc_pixel_ab themselves.
def test_step_policy_B_is_eq21_to_24_by_hand():
    # Eq. 21-24: dl_1 = eps/(|K^1|+delta), dl_2 = eps min(x2, 1-x2)/(|K^2|+delta),
    # dl_3 = eps/(|K^phi|+delta), dl = 1/(1/dl_1 + 1/dl_2 + 1/dl_3).  delta = 1e-40 is invisible in double.
    o = orc.Oracle(vac(a=0.9375, h=0.3, step_policy=1, eps=0.03, delta=1e-40))
    K = [7.7, 0.5, -0.25, 0.1]                               # K^t must not enter
    # x2 = 0.2: 1/dl = (0.5 + 0.25/0.2 + 0.1)/0.03
    assert o.step_size([0.0, 2.0, 0.2, 1.0], K) == pytest.approx(0.03 / (0.5 + 1.25 + 0.1), rel=1e-14)
    # x2 = 0.7: min(x2, 1 - x2) = 0.3 (dropping the min gives 0.03/(0.5 + 0.25/0.7 + 0.1): different by 34 %)
    assert o.step_size([0.0, 2.0, 0.7, 1.0], K) == pytest.approx(0.03 / (0.5 + 0.25 / 0.3 + 0.1), rel=1e-14)
    # beyond the pole the coordinate is folded back into [0, 1]: x2 = 1.3 -> 0.7, x2 = -0.2 -> 0.2
    assert o.step_size([0.0, 2.0, 1.3, 1.0], K) == pytest.approx(0.03 / (0.5 + 0.25 / 0.3 + 0.1), rel=1e-13)
    assert o.step_size([0.0, 2.0, -0.2, 1.0], K) == pytest.approx(0.03 / (0.5 + 1.25 + 0.1), rel=1e-13)
    # harmonic, not arithmetic, sum: one dominant component sets the step; signs do not matter; linear in eps
    assert o.step_size([0.0, 2.0, 0.5, 1.0], [1.0, -3.0, 0.0, 0.0]) == pytest.approx(0.03 / 3.0, rel=1e-13)
    assert o.step_size([0.0, 2.0, 0.5, 1.0], [1.0, 0.0, 0.0, -2.0]) == pytest.approx(0.03 / 2.0, rel=1e-13)
    o2 = orc.Oracle(vac(a=0.9375, h=0.3, step_policy=1, eps=0.06, delta=1e-40))
    assert o2.step_size([0.0, 2.0, 0.2, 1.0], K) == pytest.approx(0.06 / 1.85, rel=1e-14)
    # delta regularises a vanishing wavevector: K = 0 gives 1/(3 delta/eps + 2 delta/eps...) finite and huge
    o3 = orc.Oracle(vac(a=0.0, h=1.0, step_policy=1, eps=0.03, delta=1e-3))
    assert o3.step_size([0.0, 2.0, 0.25, 0.0], [1.0, 0.0, 0.0, 0.0]) == pytest.approx(0.03 / (1e-3 + 1e-3 / 0.25 + 1e-3), rel=1e-13)


def test_step_policy_A_clamp_and_polar_guard_by_hand():
    # BASELINE.json configs[0]: h = 0.05 (r - r_H) clamped to [1e-3, 1]; [A6] adds h <= eps_polar r |sin theta|
    # floored at 1e-3.  theta = pi x2 for h = 1.
    a = 0.9375
    rH = 1.0 + math.sqrt(1.0 - a * a)
    o = orc.Oracle(vac(a=a, h=1.0))                          # eps_polar = 0.125 (default)
    K = [1.0, 0.1, 0.1, 0.1]                                 # policy A does not look at K
    eq = 0.5                                                 # x2 = 1/2: the equator, guard inactive
    assert o.step_size([0, math.log(1000.0), eq, 0], K) == 1.0                                    # upper clamp
    assert o.step_size([0, math.log(21.0 + rH), eq, 0], K) == pytest.approx(1.0, rel=1e-12)       # 0.05 * 21 > 1
    assert o.step_size([0, math.log(3.0), eq, 0], K) == pytest.approx(0.05 * (3.0 - rH), rel=1e-13)
    assert o.step_size([0, math.log(1.4), eq, 0], K) == pytest.approx(0.05 * (1.4 - rH), rel=1e-12)
    assert o.step_size([0, math.log(rH + 0.01), eq, 0], K) == 1e-3                                # lower clamp
    # the horizon radius enters: Schwarzschild r_H = 2
    o0 = orc.Oracle(vac(a=0.0, h=1.0))
    assert o0.step_size([0, math.log(6.0), eq, 0], K) == pytest.approx(0.05 * 4.0, rel=1e-13)
    # polar guard at theta = 0.01 rad: on -> 0.125 r sin(0.01); off (eps_polar = 1e30) -> the radial rule alone
    x2 = 0.01 / math.pi
    for r in (1000.0, 8.0):
        radial = min(max(0.05 * (r - rH), 1e-3), 1.0)
        assert o.step_size([0, math.log(r), x2, 0], K) == pytest.approx(min(radial, 0.125 * r * math.sin(0.01)), rel=1e-12)
        assert o.step_size([0, math.log(r), 1.0 - x2, 0], K) == pytest.approx(min(radial, 0.125 * r * math.sin(0.01)), rel=1e-9)
    off = orc.Oracle(vac(a=a, h=1.0, eps_polar=1e30))
    assert off.step_size([0, math.log(8.0), x2, 0], K) == pytest.approx(0.05 * (8.0 - rH), rel=1e-13)
    # the guard is floored at step_min as well, and uses |sin|: beyond the pole (x2 < 0) it is still positive
    assert o.step_size([0, math.log(3.0), 1e-6, 0], K) == 1e-3
    assert o.step_size([0, math.log(8.0), -x2, 0], K) == pytest.approx(0.125 * 8.0 * math.sin(0.01), rel=1e-9)
    # other constants of the rule are parameters
    o5 = orc.Oracle(vac(a=a, h=1.0, step_c=0.02, step_min=0.01, step_max=0.25))
    assert o5.step_size([0, math.log(5.0), eq, 0], K) == pytest.approx(0.02 * (5.0 - rH), rel=1e-13)
    assert o5.step_size([0, math.log(500.0), eq, 0], K) == 0.25 and o5.step_size([0, math.log(1.4), eq, 0], K) == 0.01


def test_pixel_centres_and_image_layout_by_hand():
    # [A4b]: alpha_ix = (ix + 1/2) fov/nx - fov/2, beta_iy likewise; image[k][iy][ix], status/nsteps [iy][ix].
    s = replace(scenes.config_C3(nx=5, n_freq=2, n1=32, n2=32), ny=3, fov_M=30.0)
    o = orc.Oracle(s)
    assert o.pixel_ab(0, 0) == pytest.approx((-15.0 + 3.0, -15.0 + 5.0), abs=1e-14)      # fov/(2 nx) = 3, fov/(2 ny) = 5
    assert o.pixel_ab(4, 2) == pytest.approx((15.0 - 3.0, 15.0 - 5.0), abs=1e-14)
    assert o.pixel_ab(2, 1) == pytest.approx((0.0, 0.0), abs=1e-14)
    assert o.pixel_ab(1, 0)[0] - o.pixel_ab(0, 0)[0] == pytest.approx(6.0, abs=1e-14)    # ix <-> alpha
    assert o.pixel_ab(0, 1)[1] - o.pixel_ab(0, 0)[1] == pytest.approx(10.0, abs=1e-14)   # iy <-> beta
    # a 6 x 4 render of an asymmetric scene (Kerr, i = 20 deg, seeded grid): every pixel equals the single ray
    # traced at the hand-computed impact parameters -- a transposed image, a missing +1/2 or swapped frequency
    # planes would all fail
    s = replace(scenes.config_C3(nx=6, n_freq=2, n1=32, n2=32), ny=4, fov_M=24.0)
    o = orc.Oracle(s)
    out = o.render()
    assert out["image"].shape == (2, 4, 6) and out["status"].shape == (4, 6)
    seen = set()
    for iy in range(4):
        for ix in range(6):
            al, be = (ix + 0.5) * 24.0 / 6 - 12.0, (iy + 0.5) * 24.0 / 4 - 12.0
            r = o.trace(al, be)
            assert np.array_equal(out["image"][:, iy, ix], r["I"]), (ix, iy)
            assert out["status"][iy, ix] == r["status"] and out["nsteps"][iy, ix] == r["nsteps"]
            seen.add(float(r["I"][0]))
    assert len(seen) == 24                                   # no two pixels alike: the comparison discriminates
    assert out["steps"] == int(out["nsteps"].sum())
    # orientation by physics: the approaching side of the prograde flow is alpha < 0 (L = -alpha sin i > 0, Eq. 25),
    # i.e. the LEFT half of every row, and it is Doppler-brighter
    c1 = orc.Oracle(replace(scenes.config_C1(8), ny=4)).render()["image"][0]
    assert c1.shape == (4, 8) and c1[:, :4].sum() > 1.2 * c1[:, 4:].sum()
    b = np.unravel_index(np.argmax(c1), c1.shape)
    assert b[1] < 4 and b[0] in (1, 2)                       # brightest pixel: left half, one of the two central rows
