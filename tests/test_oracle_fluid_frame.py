"""Pins of the oracle's fluid-frame block taken THROUGH orc_transfer / orc_trace_ray.

What is pinned, each against special relativity or a Schwarzschild closed form typed here by hand (no value comes
from the oracle's own route to it, none from the CUDA path):

F1  pitch angle [A11] (the angle between k^mu and b^mu in the fluid frame) for a fluid at rest in
    flat space: the Euclidean angle between the photon direction and the field;
F2  the same for a moving fluid: relativistic aberration, cos th' = (mu - beta)/(1 - beta mu) for a field along the
    velocity, cos th' = (n.B)/(gamma (1 - beta mu)) for a field across it, and |b| = B resp. B/gamma (ideal MHD);
F3  nu = nu_hat nu_k entering Eq. 42-45 (Eq. 31, PAPER.md:180 -> PAPER.md:283-315), nu_hat = gamma (1 - beta mu) in
    flat space, (1 - 2/r)^(-1/2) for a static emitter and an E = 1 photon in Schwarzschild; dtau = nu_hat alpha L h
    (Eq. 36) and dI = j/nu_hat^2 L h w(dtau) (Eq. 35-37) with j, B_nu from the separately pinned
    orc_emissivity / orc_planck (tests/test_oracle_transfer.py P11);
F4  field directions of BASELINE.json configs[0]/[1]: radial for SPHERE (so a radial ray sees pitch angle 0 and no
    emission), toroidal for TORUS;
F5  the sampling guard of O4 / [A7]: a point outside [1.01 r_H, 1.1 r_cam] contributes nothing, so a ray through
    plasma that fills space is sampled on every step but its last.
"""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1801_10452_b200 import scenes

C_, G_, ME_, MP_ = 2.99792458e10, 6.6743e-8, 9.1093837e-28, 1.67262192e-24

R_PT, TH_PT, PH_PT = 7.0, 0.35 * math.pi, 0.9          # where the uniform scene is probed
RHO, UU, B_CODE = 1.3, 0.085, 0.07                     # primitives of the uniform fluid (code units)
NU_K = (86e9, 230e9, 1.2e12)


def _unit(v):
    v = np.asarray(v, dtype=float)
    return v / math.sqrt(v @ v)


def _to_mks(v_orth):
    """Components (r^, th^, ph^) of a vector at the probe point -> coordinate components (x1, x2, phi) of the flat
    chart r = exp(x1), theta = pi x2 (mks_h = 1, mks_r0 = 0): e_r^ = (1/r) d_x1, e_th^ = 1/(pi r) d_x2, e_ph^ = 1/(r sin th) d_phi."""
    return np.array([v_orth[0] / R_PT, v_orth[1] / (math.pi * R_PT), v_orth[2] / (R_PT * math.sin(TH_PT))])


def _uniform_scene(gamma_beta_orth, B_orth):
    """Flat space (mass 0); every cell of a GRID2D holds the same primitives, so the bilinear sampler returns them
    exactly anywhere.  The velocity and the field are chosen in the orthonormal frame AT THE PROBE POINT."""
    n1, n2 = 4, 4
    cell = np.concatenate([[RHO, UU], _to_mks(gamma_beta_orth), _to_mks(B_orth)])
    grid = np.tile(cell, (n1, n2, 1, 1))
    return scenes.Scene(name="uniform", a=0.0, mass=0.0, mks_h=1.0, mks_r0=0.0, r_cam=50.0, incl_deg=60.0,
                        plasma_model=scenes.GRID2D, M_unit_g=scenes._M_UNIT_GRID, freq_hz=NU_K,
                        n1=n1, n2=n2, n3=1, nt=1, grid_dtype=scenes.F64, x1_min=0.0, x1_max=math.log(100.0), grid=grid)


def _expected(scene, nu_hat, sin_pitch, b_code, h):
    """dI_k, dtau_k of one step of length h from Eq. 31, 35-37, 42-46 with the hand values of nu_hat, the pitch
    angle and |b|; the unit scaling (Eq. 46) typed out."""
    L = G_ * scene.M_bh_g / C_ ** 2
    rho0 = scene.M_unit_g / L ** 3
    n_e = RHO * rho0 / (MP_ + ME_)
    theta_e = (MP_ / ME_) * (scene.gamma_ad - 1.0) * (UU / RHO) / (1.0 + scene.tp_over_te)
    B_gauss = b_code * C_ * math.sqrt(4.0 * math.pi * rho0)
    dI, dtau = [], []
    for nu_k in scene.freq_hz:
        nu = nu_hat * nu_k                                           # Eq. 31
        j = orc.emissivity(nu, n_e, theta_e, B_gauss, sin_pitch)
        alpha = j / orc.planck(nu, theta_e) if j > 0 else 0.0        # Kirchhoff
        dt = nu_hat * alpha * L * h                                  # Eq. 36
        w = -math.expm1(-dt) / dt if dt > 0 else 1.0
        dI.append(j / nu_hat ** 2 * L * h * w)
        dtau.append(dt)
    return np.array(dI), np.array(dtau)


def _photon(n_orth):
    X = [0.0, math.log(R_PT), TH_PT / math.pi, PH_PT]
    K = [1.0] + list(_to_mks(n_orth))                                # k^t = 1: unit energy in the lab frame
    return X, K


# --------------------------------------------------------------------------------------- F1
@pytest.mark.parametrize("psi", [0.02, 0.7, 0.5 * math.pi, 2.4])
def test_F1_pitch_angle_of_a_fluid_at_rest_is_the_euclidean_angle(psi):
    e_B = _unit([0.3, -0.5, 0.8])
    e_perp = _unit(np.cross(e_B, [1.0, 0.2, -0.4]))
    n = math.cos(psi) * e_B + math.sin(psi) * e_perp                 # photon direction at angle psi to the field
    s = _uniform_scene([0.0, 0.0, 0.0], B_CODE * e_B)
    o = orc.Oracle(s)
    X, K = _photon(n)
    assert abs(o.null_norm(X, K)) < 1e-14
    h = 0.37
    ok, I, tau = o.transfer(X, K, h, np.zeros(3), np.zeros(3))
    assert ok == 1
    dI, dtau = _expected(s, 1.0, math.sin(psi), B_CODE, h)
    assert np.all(dI > 0)
    np.testing.assert_allclose(I, dI, rtol=1e-8)
    np.testing.assert_allclose(tau, dtau, rtol=1e-8)
    # and the update attenuates by the optical depth already behind the point (Eq. 37): I += dI exp(-tau)
    ok, I2, tau2 = o.transfer(X, K, h, np.full(3, 2e-6), np.array([0.5, 1.5, 0.0]))
    np.testing.assert_allclose(I2 - 2e-6, dI * np.exp(-np.array([0.5, 1.5, 0.0])), rtol=1e-7)
    np.testing.assert_allclose(tau2 - np.array([0.5, 1.5, 0.0]), dtau, rtol=1e-8, atol=1e-16)


# ---------------------------------------------------------------------------------- F2, F3
@pytest.mark.parametrize("beta", [0.6, 0.95])
@pytest.mark.parametrize("mu", [-0.8, 0.1, 0.9])
def test_F2_F3_moving_fluid_doppler_shift_and_aberrated_pitch_angle(beta, mu):
    gam = 1.0 / math.sqrt(1.0 - beta * beta)
    e_v = _unit([-0.4, 0.7, 0.5])
    e_1 = _unit(np.cross(e_v, [0.1, 1.0, 0.3]))
    e_2 = np.cross(e_v, e_1)
    chi = 0.6
    n = mu * e_v + math.sqrt(1 - mu * mu) * (math.cos(chi) * e_1 + math.sin(chi) * e_2)
    X, K = _photon(n)
    nu_hat = gam * (1.0 - beta * mu)                                 # Doppler factor of a photon of lab energy 1
    h = 0.21
    # field along the velocity: unchanged by the boost, pitch angle by the aberration formula
    s = _uniform_scene(gam * beta * e_v, B_CODE * e_v)
    o = orc.Oracle(s)
    pl = o.plasma(X)
    assert pl["u"][0] == pytest.approx(gam, rel=1e-12)
    cos_p = (mu - beta) / (1.0 - beta * mu)
    ok, I, tau = o.transfer(X, K, h, np.zeros(3), np.zeros(3))
    dI, dtau = _expected(s, nu_hat, math.sqrt(1 - cos_p * cos_p), B_CODE, h)
    assert ok == 1 and np.all(dI > 0)
    np.testing.assert_allclose(I, dI, rtol=1e-8)
    np.testing.assert_allclose(tau, dtau, rtol=1e-8)
    # field across the velocity (ideal MHD: E' = 0): |b| = B/gamma, direction kept, n'_perp = n_perp / nu_hat
    s = _uniform_scene(gam * beta * e_v, B_CODE * e_1)
    o = orc.Oracle(s)
    cos_p = float(n @ e_1) / nu_hat
    ok, I, tau = o.transfer(X, K, h, np.zeros(3), np.zeros(3))
    dI, dtau = _expected(s, nu_hat, math.sqrt(1 - cos_p * cos_p), B_CODE / gam, h)
    assert ok == 1 and np.all(dI > 0)
    np.testing.assert_allclose(I, dI, rtol=1e-8)
    np.testing.assert_allclose(tau, dtau, rtol=1e-8)
    # the Doppler shift is not a detail: without it the 1.2 THz emissivity would be off by far more than the bar
    static, _ = _expected(s, 1.0, math.sqrt(1 - cos_p * cos_p), B_CODE / gam, h)
    assert abs(static[2] / dI[2] - 1.0) > 1e-3


def test_F3_gravitational_redshift_enters_emissivity_and_optical_depth():
    """Static slab in Schwarzschild: u = (-g_tt)^(-1/2) d_t and E = -k_t = 1 give nu_hat = (1 - 2/r)^(-1/2)."""
    sin_pitch = 0.6
    s = scenes.slab_scene(2e4, 8.0, 25.0, 9.0, sin_pitch=sin_pitch, nu_hz=230e9, mass=1.0, r_cam=60.0, incl_deg=40.0)
    s = replace(s, freq_hz=(230e9, 690e9))
    o = orc.Oracle(s)
    picks = []
    for (alpha, beta), pick in (((5.0, 4.0), np.argmin), ((3.0, 9.0), np.argmax)):     # b > sqrt(27): both escape
        res = o.trace(alpha, beta, record_path=True)
        assert res["status"] == 2
        path = res["path"]
        r = np.exp(path[:, 1])
        z = r * np.cos(math.pi * path[:, 2])
        inside = np.nonzero(np.abs(z) < 4.4)[0]
        i = inside[pick(r[inside])]
        picks.append((path[i, :4], path[i, 4:], r[i]))
    assert picks[0][2] < 5.0 and picks[1][2] > 11.0                  # one point deep in the well, one further out
    L = G_ * s.M_bh_g / C_ ** 2
    for X, K, r_i in picks:
        nu_hat = 1.0 / math.sqrt(1.0 - 2.0 / r_i)
        h = 0.11
        ok, I, tau = o.transfer(X, K, h, np.zeros(2), np.zeros(2))
        assert ok == 1
        for k, nu_k in enumerate(s.freq_hz):
            nu = nu_hat * nu_k
            j = orc.emissivity(nu, 2e4, 8.0, 25.0, sin_pitch)
            dt = nu_hat * (j / orc.planck(nu, 8.0)) * L * h
            assert tau[k] == pytest.approx(dt, rel=1e-5)          # E = 1 holds to the RK4 error of the path (~1e-7)
            assert I[k] == pytest.approx(j / nu_hat ** 2 * L * h * (-math.expm1(-dt) / dt), rel=1e-5)
            # a dropped shift would be visible: j(nu_k) differs from j(nu_hat nu_k) by much more than the bar
            assert abs(orc.emissivity(nu_k, 2e4, 8.0, 25.0, sin_pitch) / j - 1.0) > 1e-3


# --------------------------------------------------------------------------------------- F4
def test_F4_sphere_field_is_radial_and_a_radial_ray_sees_no_emission():
    o = orc.Oracle(scenes.config_C0(8))
    for X in ([0.0, math.log(3.0), 0.31, 0.4], [2.0, math.log(40.0), 0.77, 5.0]):
        p = o.plasma(X)["p"]
        assert p[2] == 0.0 and p[3] == 0.0 and p[1] > 0.0            # along d_x1 (plus a d_t part from the projection)
    # alpha = beta = 0 in Schwarzschild is the radial ray: k, u and b all radial, pitch angle 0, nu_s = 0, j = 0 [A13]
    centre = o.trace(0.0, 0.0)
    side = o.trace(6.0, 0.0)
    assert centre["status"] == 1 and centre["nsampled"] > 100
    assert side["I"][0] > 0.0
    assert centre["I"][0] < 1e-12 * side["I"][0]
    assert centre["tau"][0] < 1e-12 * side["tau"][0]


def test_F4_torus_field_is_toroidal():
    o = orc.Oracle(scenes.config_C1(8))
    for X in ([0.0, math.log(12.0), 0.5, 0.0], [1.0, math.log(9.0), 0.46, 2.0]):
        pl = o.plasma(X)
        p = pl["p"]
        assert p[1] == 0.0 and p[2] == 0.0 and p[3] > 0.0            # along d_phi (plus a d_t part)
    # a photon moving along the field in the fluid frame (k = nu (u + b^)) has pitch angle 0: no emission;
    # one moving along the polar direction (orthogonal to u and b in this axisymmetric flow) has pitch angle 90 deg
    X = [0.0, math.log(12.0), 0.5, 0.0]
    pl = o.plasma(X)
    g = o.metric(X)
    b_hat = pl["p"] / math.sqrt(pl["p"] @ g @ pl["p"])
    e_th = np.array([0.0, 0.0, 1.0, 0.0]) / math.sqrt(g[2, 2])
    assert abs(e_th @ g @ pl["u"]) < 1e-14 and abs(e_th @ g @ b_hat) < 1e-14
    ok, I_par, _ = o.transfer(X, pl["u"] + b_hat, 0.1, [0.0], [0.0])
    ok, I_perp, _ = o.transfer(X, pl["u"] + e_th, 0.1, [0.0], [0.0])
    ok, I_45, _ = o.transfer(X, pl["u"] + (b_hat + e_th) / math.sqrt(2.0), 0.1, [0.0], [0.0])
    j90 = orc.emissivity(230e9, pl["n_e"], pl["theta_e"], pl["B"], 1.0)
    j45 = orc.emissivity(230e9, pl["n_e"], pl["theta_e"], pl["B"], math.sqrt(0.5))
    Lh = G_ * o.scene.M_bh_g / C_ ** 2 * 0.1
    assert I_perp[0] == pytest.approx(j90 * Lh, rel=1e-6)            # nu_hat = 1 for these photons; optically thin
    assert I_45[0] == pytest.approx(j45 * Lh, rel=1e-6)
    assert I_par[0] < 1e-12 * I_perp[0]


# --------------------------------------------------------------------------------------- F5
def test_F5_points_outside_the_radial_range_are_not_sampled():
    o = orc.Oracle(scenes.config_C0(8))                               # the sphere fills space: plasma at every point
    rH = 2.0
    for alpha, beta, status in ((8.0, 3.0, 2), (1.0, 0.5, 1)):
        res = o.trace(alpha, beta, record_path=True)
        assert res["status"] == status
        r = np.exp(res["path"][:, 1])
        outside = (r < 1.01 * rH) | (r > 1.1 * o.scene.r_cam)
        assert outside.sum() == 1 and outside[-1]                    # only the last point left the range ([A7])
        assert res["nsampled"] == res["nsteps"] - 1
    # and the transfer on the captured ray's last point would not have been nothing: the guard is what keeps it out
    X, K = res["path"][-1, :4], res["path"][-1, 4:]
    ok, I, tau = o.transfer(X, K, 1.0, [0.0], [0.0])
    assert ok == 1 and I[0] > 0.0
