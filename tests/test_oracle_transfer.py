"""Pins of the oracle's plasma sampler and radiative transfer against closed forms, the paper's
printed numbers and direct quadrature -- no expected value comes from the oracle or the CUDA path.

P8  uniform slab: I = j L (thin), I = S (1 - exp(-tau)) (any step), I -> B_nu (thick)
P9  backward integration (Eq. 37) equals the forward formal solution (Eq. 35) on the same samples
P11 Eq. 42-45: fit vs direct quadrature over the Maxwell-Juettner distribution (Eq. 41), the
    cyclotron frequency the paper prints, Kirchhoff, Rayleigh-Jeans limit
P12 multilinear interpolation: exactness, continuity, periodicity, slow light == fast light on
    identical snapshots
plus: four-velocity normalisation, b.u = 0, unit scaling (Eq. 46), plasma beta of the models.
"""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1801_10452_b200 import scenes

# CGS constants typed independently of the oracle (CODATA 2018)
C_, E_, ME_, MP_, KB_, H_ = 2.99792458e10, 4.80320471e-10, 9.1093837e-28, 1.67262192e-24, 1.380649e-16, 6.62607015e-27


# ------------------------------------------------------------------------------------ P11
def test_P11_cyclotron_frequency_printed_in_the_paper(golden):
    # nu_s = (2/9) nu_c Theta^2 sin(theta) (Eq. 44) enters j only through X = nu/nu_s: recover nu_c from
    # the position of the maximum of X-dependence?  Simpler: j is proportional to nu_s * F(nu/nu_s); for two
    # field strengths B1, B2 = 2 B1 and nu2 = 2 nu1 the ratio j2/j1 must be exactly 2 (same X).
    j1 = orc.emissivity(1e11, 1.0, 3.0, 10.0, 0.5)
    j2 = orc.emissivity(2e11, 1.0, 3.0, 20.0, 0.5)
    assert j2 / j1 == pytest.approx(2.0, rel=1e-13)
    # and the constant itself: e/(2 pi m_e c) = 2.8e6 Hz/G as printed
    assert E_ / (2 * math.pi * ME_ * C_) == pytest.approx(golden["nu_c_per_gauss"], rel=2e-3)


def _j_direct(nu, n_e, theta_e, B, theta):
    """Thermal synchrotron emissivity by direct quadrature: single-electron power
    P(nu) = sqrt(3) e^3 B sin(th)/(m c^2) F(nu/nu_cr), nu_cr = 3/2 gamma^2 nu_c sin(th),
    F(x) = x int_x^inf K_{5/3}, averaged over Eq. 41 (Maxwell-Juettner), j = P/(4 pi)."""
    from scipy import integrate, special

    nu_c = E_ * B / (2 * math.pi * ME_ * C_)

    def F(x):
        if x > 600:
            return 0.0
        val, _ = integrate.quad(lambda t: special.kv(5.0 / 3.0, t), x, np.inf, limit=200)
        return x * val

    k2 = special.kn(2, 1.0 / theta_e)

    def integrand(gam):
        dist = gam * math.sqrt(gam * gam - 1.0) * math.exp(-gam / theta_e) / (theta_e * k2)    # Eq. 41 / n_e
        x = nu / (1.5 * gam * gam * nu_c * math.sin(theta))
        return dist * F(x)

    val, _ = integrate.quad(integrand, 1.0, 1.0 + 80.0 * theta_e, limit=400)
    return n_e * math.sqrt(3.0) * E_ ** 3 * B * math.sin(theta) / (4 * math.pi * ME_ * C_ ** 2) * val


@pytest.mark.parametrize("theta_e,ratio", [(10.0, 1e4), (10.0, 1e5), (3.0, 1e4), (1.0, 1e2), (1.0, 1e3), (3.0, 1e2),
                                           (3.0, 1e3), (10.0, 1e2), (10.0, 1e3), (30.0, 1e3)])
def test_P11_emissivity_fit_against_direct_quadrature(theta_e, ratio, golden):
    # < 1 % for Theta_e > 0.5, nu/nu_c > 10 at theta = 30 deg.  (A prefactor sqrt(2 pi)
    # instead of sqrt(2) pi -- the garbled print of Eq. 42 -- would be off by 44 %.)
    # k2_mode = 1 evaluates K_2 exactly as Eq. 41-42 are written; the 2 Theta^2 shortcut is tested below.
    # Measured fit error (fit/quadrature - 1) at 30 deg, recorded in DESIGN.md 3.4: +0.2 % ... +2.3 % over
    # Theta_e in [1, 30], nu/nu_c in [1e2, 1e5] (largest at Theta_e >= 10, nu/nu_c = 1e2); the paper's "< 1 %" holds
    # for nu/nu_c >= 1e3 at Theta_e <= 3 and nu/nu_c >= 1e4 at Theta_e = 10, hence the bar of 3 x its bound here.
    B, th = 30.0, math.radians(golden["fit_theta_deg"])
    nu = ratio * E_ * B / (2 * math.pi * ME_ * C_)
    j_fit = orc.emissivity(nu, 1e6, theta_e, B, math.sin(th), k2_mode=1)
    j_num = _j_direct(nu, 1e6, theta_e, B, th)
    assert j_fit == pytest.approx(j_num, rel=3 * golden["fit_error_bound"])


def test_P11_bessel_k2_and_the_2theta2_shortcut():
    from scipy import special
    for x in (0.05, 0.3, 1.0, 4.0):
        assert orc.bessel_k2(x) == pytest.approx(special.kn(2, x), rel=1e-10)
    # K_2(1/Theta) -> 2 Theta^2 for Theta >> 1: "differences ... of a few percent at most"
    for theta_e in (5.0, 20.0, 100.0):
        j0 = orc.emissivity(2.3e11, 1e6, theta_e, 30.0, 0.7, k2_mode=0)
        j1 = orc.emissivity(2.3e11, 1e6, theta_e, 30.0, 0.7, k2_mode=1)
        assert j0 / j1 == pytest.approx(special.kn(2, 1 / theta_e) / (2 * theta_e ** 2), rel=1e-9)
        assert abs(j0 / j1 - 1) < 0.03


def test_P11_planck_function_limits():
    for nu, theta_e in [(1e9, 10.0), (2.3e11, 3.0), (1e13, 0.5)]:
        T = theta_e * ME_ * C_ ** 2 / KB_
        x = H_ * nu / (KB_ * T)
        expect = 2 * H_ * nu ** 3 / C_ ** 2 / math.expm1(x)
        assert orc.planck(nu, theta_e) == pytest.approx(expect, rel=1e-13)
    # Rayleigh-Jeans: B_nu -> 2 nu^2 k T / c^2 for h nu << k T
    T = 10.0 * ME_ * C_ ** 2 / KB_
    assert orc.planck(1e8, 10.0) == pytest.approx(2 * 1e16 * KB_ * T / C_ ** 2, rel=1e-9)


def test_P11_emissivity_degenerate_cases():
    assert orc.emissivity(2.3e11, 1e6, 10.0, 30.0, 0.0) == 0.0            # along the field
    assert orc.emissivity(2.3e11, 0.0, 10.0, 30.0, 0.5) == 0.0            # no electrons
    assert orc.emissivity(2.3e11, 1e6, 10.0, 0.0, 0.5) == 0.0             # no field
    # j -> 0 smoothly as sin(theta) -> 0
    js = [orc.emissivity(2.3e11, 1e6, 10.0, 30.0, s) for s in (1e-2, 1e-3, 1e-4, 1e-6)]
    assert all(a > b >= 0.0 for a, b in zip(js, js[1:]))


# ------------------------------------------------------------------------------------- P8
def test_P8_transfer_update_telescopes_to_the_formal_solution():
    # uniform medium, arbitrary unequal steps: I = S (1 - exp(-tau)) exactly (Eq. 35), S = j/alpha
    rng = np.random.default_rng(7)
    j, alpha, nu_hat, Lcm = 3e-18, 2e-13, 1.7, 6.6e11
    I, tau, length = 0.0, 0.0, 0.0
    for h in rng.uniform(0.01, 2.0, size=40):
        I, tau = orc.transfer_update(I, tau, j, alpha, nu_hat, Lcm, h)
        length += h
    tau_expect = nu_hat * alpha * Lcm * length
    assert tau == pytest.approx(tau_expect, rel=1e-13)
    S = j / alpha / nu_hat ** 3          # invariant source function times nu_obs^3 (nu_obs = 1 unit)
    assert I == pytest.approx(S * (1 - math.exp(-tau_expect)), rel=1e-12)
    # optically thin limit of the same formula: I = j L / nu_hat^2
    I2, tau2 = orc.transfer_update(0.0, 0.0, j, 1e-30, nu_hat, Lcm, 1.0)
    assert I2 == pytest.approx(j * Lcm / nu_hat ** 2, rel=1e-12)
    # alpha = 0 exactly takes the w = 1 branch
    I3, tau3 = orc.transfer_update(0.0, 0.0, j, 0.0, nu_hat, Lcm, 1.0)
    assert tau3 == 0.0 and I3 == pytest.approx(j * Lcm / nu_hat ** 2, rel=1e-15)


def _slab_intensity(n_e, thickness, step_max=0.02, nu=230e9, theta_e=10.0, B=30.0):
    s = scenes.slab_scene(n_e, theta_e, B, thickness, sin_pitch=1.0, nu_hz=nu, step_c=0.0, step_min=step_max,
                          step_max=step_max, eps_polar=1e30, r_cam=60.0, incl_deg=30.0)
    o = orc.Oracle(s)
    res = o.trace(4.0, 3.0)
    assert res["status"] == 2
    return o, res


def test_P8_optically_thin_slab_gives_j_times_path_length():
    thickness, inc = 8.0, math.radians(30.0)
    o, res = _slab_intensity(1e-5, thickness, step_max=0.02)
    j = orc.emissivity(230e9, 1e-5, 10.0, 30.0, 1.0)
    assert 0 < res["tau"][0] < 1e-10
    # all rays leave the camera point, so the ray direction differs from the inclination by ~b/r_cam;
    # measure the chord through |z| < thickness/2 from the traced path itself
    path = o.trace(4.0, 3.0, record_path=True)["path"]
    z = np.exp(path[:, 1]) * np.cos(math.pi * path[:, 2])
    inside = np.abs(z) < thickness / 2
    assert res["nsampled"] == inside.sum()
    L_path = inside.sum() * 0.02
    assert L_path == pytest.approx(thickness / math.cos(inc), rel=0.05)           # b/r_cam = 5/60 rad off axis
    assert res["I"][0] == pytest.approx(j * L_path * o.scene.L_cm, rel=1e-10)       # I = j L  (nu_hat = 1)


def test_P8_slab_of_any_depth_follows_S_one_minus_exp_minus_tau():
    for n_e in (3e5, 3e6):
        o, res = _slab_intensity(n_e, 8.0, step_max=0.05)
        tau = res["tau"][0]
        assert 0.01 < tau < 50
        S = orc.planck(230e9, 10.0)                                      # Kirchhoff: S = j/alpha = B_nu
        assert res["I"][0] == pytest.approx(S * (1 - math.exp(-tau)), rel=1e-11)


def test_P8_optically_thick_slab_saturates_at_the_planck_function():
    o, res = _slab_intensity(1e9, 8.0, step_max=0.05)
    assert res["tau"][0] > 100
    T = 10.0 * ME_ * C_ ** 2 / KB_
    B_nu = 2 * H_ * 230e9 ** 3 / C_ ** 2 / math.expm1(H_ * 230e9 / (KB_ * T))
    assert res["I"][0] == pytest.approx(B_nu, rel=1e-12)


# ------------------------------------------------------------------------------------- P9
def test_P9_backward_equals_forward_formal_solution_and_is_monotone():
    s = scenes.config_C3(nx=8, n_freq=4, n1=48, n2=48)
    o = orc.Oracle(s)
    al, be = 6.0, 1.5
    res = o.trace(al, be, record_path=True)
    path = res["path"]
    # per-step contributions: transfer from (I, tau) = 0 returns dI0 = S (1 - exp(-dtau)) and dtau
    X0, K0 = o.camera(al, be)
    hs, Xprev, Kprev = [], X0, K0
    dI, dtau = [], []
    for row in path:
        hs.append(o.step_size(Xprev, Kprev))
        ok, I1, t1 = o.transfer(row[:4], row[4:], hs[-1], np.zeros(4), np.zeros(4))
        dI.append(I1 if ok else np.zeros(4))
        dtau.append(t1 if ok else np.zeros(4))
        Xprev, Kprev = row[:4], row[4:]
    dI, dtau = np.array(dI), np.array(dtau)
    assert (dtau.sum(0) > 0).all() and res["nsampled"] > 50
    # forward: from the far end toward the camera, Eq. 35 per step
    I_fwd = np.zeros(4)
    for n in range(len(path) - 1, -1, -1):
        I_fwd = I_fwd * np.exp(-dtau[n]) + dI[n]
    assert np.allclose(I_fwd, res["I"], rtol=1e-11, atol=0)
    # backward partial sums are monotone non-decreasing
    partial = np.cumsum(dI * np.exp(-np.vstack([np.zeros(4), np.cumsum(dtau, 0)[:-1]])), 0)
    assert (np.diff(partial, axis=0) >= 0).all()
    assert np.allclose(partial[-1], res["I"], rtol=1e-11)
    assert np.allclose(dtau.sum(0), res["tau"], rtol=1e-11)
    # spectrum sanity: thick at 1e9 Hz, thin at 1e16 Hz
    assert res["tau"][0] > 10 * res["tau"][-1]


# ------------------------------------------------------------------------ plasma samplers
@pytest.mark.parametrize("cfg", ["C0", "C1", "C2", "C4"])
def test_plasma_four_velocity_and_field_direction(cfg):
    if cfg == "C0":
        s = scenes.config_C0(8)
    elif cfg == "C1":
        s = scenes.config_C1(8)
    elif cfg == "C2":
        s = scenes.config_C2(nx=8, n1=32, n2=32)
    else:
        s = scenes.config_C4(nx=8, n1=16, n2=12, n3=8, nt=4)
    o = orc.Oracle(s)
    rng = np.random.default_rng(3)
    n_present = 0
    for _ in range(60):
        X = [rng.uniform(0, 30), rng.uniform(math.log(1.5), math.log(30.0)), rng.uniform(0.05, 0.95), rng.uniform(0, 6.28)]
        pl = o.plasma(X)
        if pl is None:
            continue
        n_present += 1
        g = o.metric(X)
        assert pl["u"] @ g @ pl["u"] == pytest.approx(-1.0, rel=1e-11)          # timelike unit
        assert abs(pl["p"] @ g @ pl["u"]) < 1e-10 * max(1.0, abs(pl["p"]).max() * abs(pl["u"]).max() * abs(g).max())
        assert pl["p"] @ g @ pl["p"] > 0                                         # spacelike
        assert pl["n_e"] > 0 and pl["theta_e"] > 0 and pl["B"] > 0 and pl["u"][0] > 0
    assert n_present > 10


def test_analytic_models_density_temperature_and_beta():
    o = orc.Oracle(scenes.config_C0(8))
    for r in (2.5, 7.0, 40.0):
        pl = o.plasma([0, math.log(r), 0.4, 0])
        n, T = 1e6 * r ** -1.5, 1e11 / r
        assert pl["n_e"] == pytest.approx(n, rel=1e-12)
        assert pl["theta_e"] == pytest.approx(KB_ * T / (ME_ * C_ ** 2), rel=1e-12)
        assert n * KB_ * T / (pl["B"] ** 2 / (8 * math.pi)) == pytest.approx(10.0, rel=1e-12)   # beta = 10
    o = orc.Oracle(scenes.config_C1(8))
    assert o.plasma([0, math.log(3.9), 0.5, 0]) is None and o.plasma([0, math.log(20.1), 0.5, 0]) is None
    pl = o.plasma([0, math.log(12.0), 0.5, 0])
    assert pl["n_e"] == pytest.approx(1e7, rel=1e-12)                         # n_e,max at r = 12 M on the equator
    th = math.pi * 0.4
    pl2 = o.plasma([0, math.log(12.0), 0.4, 0])
    assert pl2["n_e"] == pytest.approx(1e7 * math.exp(-math.cos(th) ** 2 / (2 * 0.3 ** 2)), rel=1e-12)
    # Keplerian: u^phi/u^t = 1/(r^1.5 + a)
    assert pl["u"][3] / pl["u"][0] == pytest.approx(1.0 / (12.0 ** 1.5 + 0.9375), rel=1e-13)
    assert pl["u"][1] == 0.0 and pl["u"][2] == 0.0


def test_grid_unit_scaling_eq46_and_electron_temperature():
    s = scenes.config_C2(nx=8, n1=32, n2=32)
    o = orc.Oracle(s)
    d1 = (s.x1_max - s.x1_min) / s.n1
    i, j = 20, 15
    X = [0.0, s.x1_min + (i + 0.5) * d1, (j + 0.5) / s.n2, 0.3]
    prim = o.grid_interp(X)
    assert np.allclose(prim, s.grid[i, j, 0], rtol=1e-14)                   # cell centre: the stored values
    pl = o.plasma(X)
    L = 6.6743e-8 * s.M_bh_g / C_ ** 2
    rho0 = s.M_unit_g / L ** 3
    assert pl["n_e"] == pytest.approx(prim[0] * rho0 / (MP_ + ME_), rel=1e-12)                    # Eq. 46
    assert pl["theta_e"] == pytest.approx((MP_ / ME_) * (s.gamma_ad - 1) * prim[1] / prim[0] / (1 + s.tp_over_te), rel=1e-12)
    # the generator's promise: rho = 1 <-> n_e = 1e7 cm^-3
    assert rho0 / (MP_ + ME_) == pytest.approx(1e7, rel=1e-12)
    # field strength: b^2 from the primitives with the metric, scaled by B0 = c sqrt(4 pi rho0)
    g = o.metric(X)
    b2 = pl["p"] @ g @ pl["p"]
    assert pl["B"] == pytest.approx(math.sqrt(b2) * C_ * math.sqrt(4 * math.pi * rho0), rel=1e-12)
    # HARM relations: u^t = gamma/alpha, b^t = g_{i mu} B^i u^mu, b^i = (B^i + b^t u^i)/u^t
    gi = o.metric_inv(X)
    alpha_l = 1 / math.sqrt(-gi[0, 0])
    ut = np.array([0, prim[2], prim[3], prim[4]])
    gam = math.sqrt(1 + ut @ g @ ut)
    assert pl["u"][0] == pytest.approx(gam / alpha_l, rel=1e-12)
    Bv = np.array([0, prim[5], prim[6], prim[7]])
    bt = Bv @ g @ pl["u"]
    assert pl["p"][0] == pytest.approx(bt, rel=1e-11)
    assert np.allclose(pl["p"][1:], (Bv[1:] + bt * pl["u"][1:]) / pl["u"][0], rtol=1e-11)


def test_electron_temperature_ratio_eq47_limits_and_reduction():
    # Eq. 47: T_p/T_e = R_low/(1+beta_p^2) + R_high beta_p^2/(1+beta_p^2), beta_p = P_gas/P_mag,
    # P_mag = b^2/2.  Pinned by what the paper states about it: beta_p << 1 -> R_low, beta_p >> 1 -> R_high
    # (PAPER.md:377), R_low = R_high = R is the constant-ratio model (the disk model of PAPER.md:399 has both = 1),
    # and beta_p = 1 gives the mean of the two.
    base = scenes.config_C2(nx=8, n1=32, n2=32)
    d1 = (base.x1_max - base.x1_min) / base.n1
    X = [0.0, base.x1_min + 20.5 * d1, 15.5 / base.n2, 0.3]
    const = orc.Oracle(base).plasma(X)

    def theta_e(grid, r_low, r_high):
        s = replace(base, te_model=1, model=(r_low, r_high) + (0.0,) * 14, grid=grid)
        return orc.Oracle(s).plasma(X)["theta_e"]

    # R_low = R_high = tp_over_te: identical to the constant-ratio path, which test_grid_unit_scaling pins
    assert theta_e(base.grid, 3.0, 3.0) == pytest.approx(const["theta_e"], rel=1e-14)
    scale = (MP_ / ME_) * (base.gamma_ad - 1)
    u_over_rho = base.grid[20, 15, 0, 1] / base.grid[20, 15, 0, 0]
    weak, strong = base.grid.copy(), base.grid.copy()
    weak[..., 5:] *= 1e-6          # b^2 -> 1e-12 b^2: beta_p >> 1
    strong[..., 5:] *= 1e3         # beta_p << 1
    assert theta_e(weak, 1.0, 25.0) == pytest.approx(scale * u_over_rho / (1 + 25.0), rel=1e-9)
    assert theta_e(strong, 1.0, 25.0) == pytest.approx(scale * u_over_rho / (1 + 1.0), rel=1e-6)
    # beta_p = 1 exactly: rescale the field so that b^2/2 = (gamma - 1) u at this cell (b^2 is quadratic in B^i)
    o = orc.Oracle(base)
    g = o.metric(X)
    b2 = const["p"] @ g @ const["p"]
    lam = math.sqrt((base.gamma_ad - 1) * base.grid[20, 15, 0, 1] / (0.5 * b2))
    unit = base.grid.copy()
    unit[..., 5:] *= lam
    assert theta_e(unit, 1.0, 25.0) == pytest.approx(scale * u_over_rho / (1 + 13.0), rel=1e-10)
    # zero field: the beta_p -> infinity limit
    zero = base.grid.copy()
    zero[..., 5:] = 0.0
    assert theta_e(zero, 1.0, 25.0) == pytest.approx(scale * u_over_rho / 26.0, rel=1e-13)


# ------------------------------------------------------------------------------------ P12
def _linear_grid_scene(n1=12, n2=10, n3=8, nt=5, slow=True):
    """A grid whose 8 fields are multilinear in (x1, x2, t) and a trig polynomial in phi."""
    s = scenes.Scene(a=0.5, mks_h=0.3, plasma_model=scenes.GRID3DT, n1=n1, n2=n2, n3=n3, nt=nt,
                     grid_dtype=scenes.F64, slow_light=1 if slow else 0, snapshot=2,
                     x1_min=math.log(1.2), x1_max=math.log(50.0), t0=5.0, dt_snap=10.0, M_unit_g=1e20)
    d1 = (s.x1_max - s.x1_min) / n1
    x1 = s.x1_min + (np.arange(n1) + 0.5) * d1
    x2 = (np.arange(n2) + 0.5) / n2
    t = s.t0 + np.arange(nt) * s.dt_snap
    ph = (np.arange(n3) + 0.5) * 2 * math.pi / n3
    T, A, B, P = np.meshgrid(t, x1, x2, ph, indexing="ij")
    g = np.empty((nt, n1, n2, n3, 8))
    for f in range(8):
        g[..., f] = (1 + f) + 0.3 * A - 0.7 * B + 0.01 * T + 0.05 * f * A * B + 0.002 * A * T
    s.grid = g
    return s


def test_P12_multilinear_fields_are_reproduced_exactly():
    s = _linear_grid_scene()
    o = orc.Oracle(s)
    rng = np.random.default_rng(5)
    d1 = (s.x1_max - s.x1_min) / s.n1
    for _ in range(50):
        A = rng.uniform(s.x1_min + 0.5 * d1, s.x1_max - 0.5 * d1)
        B = rng.uniform(0.5 / s.n2, 1 - 0.5 / s.n2)
        T = rng.uniform(s.t0, s.t0 + (s.nt - 1) * s.dt_snap)
        prim = o.grid_interp([T, A, B, rng.uniform(-10, 10)])
        for f in range(8):
            assert prim[f] == pytest.approx((1 + f) + 0.3 * A - 0.7 * B + 0.01 * T + 0.05 * f * A * B + 0.002 * A * T, rel=1e-13)
    # outside the radial range: absent; time clamps to the first / last snapshot
    assert o.grid_interp([10.0, s.x1_min + 0.4 * d1, 0.5, 0.0]) is None
    assert o.grid_interp([10.0, s.x1_max - 0.4 * d1, 0.5, 0.0]) is None
    lo, lo2 = o.grid_interp([-1e9, 1.0, 0.5, 0.0]), o.grid_interp([s.t0, 1.0, 0.5, 0.0])
    assert np.array_equal(lo, lo2)
    hi, hi2 = o.grid_interp([1e9, 1.0, 0.5, 0.0]), o.grid_interp([s.t0 + (s.nt - 1) * s.dt_snap, 1.0, 0.5, 0.0])
    assert np.array_equal(hi, hi2)


def test_P12_phi_periodicity_pole_fold_and_continuity():
    s = scenes.config_C4(nx=8, n1=16, n2=12, n3=8, nt=4)
    o = orc.Oracle(s)
    X = [12.0, 1.7, 0.37, 1.234]
    base = o.grid_interp(X)
    assert np.allclose(o.grid_interp([12.0, 1.7, 0.37, 1.234 + 2 * math.pi]), base, rtol=1e-12)
    assert np.allclose(o.grid_interp([12.0, 1.7, 0.37, 1.234 - 4 * math.pi]), base, rtol=1e-12)
    # across the periodic seam phi = 0 and across cell faces: continuous
    for e in (1e-9,):
        assert np.allclose(o.grid_interp([12.0, 1.7, 0.37, -e]), o.grid_interp([12.0, 1.7, 0.37, e]), rtol=1e-7)
        dphi = 2 * math.pi / s.n3
        assert np.allclose(o.grid_interp([12.0, 1.7, 0.37, 1.5 * dphi - e]), o.grid_interp([12.0, 1.7, 0.37, 1.5 * dphi + e]), rtol=1e-7)
        assert np.allclose(o.grid_interp([12.0, 1.7, 2.5 / s.n2 - e, 1.0]), o.grid_interp([12.0, 1.7, 2.5 / s.n2 + e, 1.0]), rtol=1e-7)
        assert np.allclose(o.grid_interp([20.0 - e, 1.7, 0.37, 1.0]), o.grid_interp([20.0 + e, 1.7, 0.37, 1.0]), rtol=1e-7)
    # pole fold: x2 -> -x2 with phi -> phi + pi (and x2 -> 2 - x2 at the south pole)
    assert np.allclose(o.grid_interp([12.0, 1.7, -0.02, 1.0]), o.grid_interp([12.0, 1.7, 0.02, 1.0 + math.pi]), rtol=1e-12)
    assert np.allclose(o.grid_interp([12.0, 1.7, 1.03, 1.0]), o.grid_interp([12.0, 1.7, 0.97, 1.0 + math.pi]), rtol=1e-12)


def test_P12_slow_light_over_identical_snapshots_is_fast_light():
    s = scenes.config_C4(nx=8, n1=16, n2=12, n3=8, nt=4)
    g = np.repeat(s.grid[2:3], 4, axis=0)                     # four copies of one snapshot
    slow = replace(s, grid=g, slow_light=1, t_cam=1000.0)
    fast = replace(s, grid=g, slow_light=0, snapshot=1, t_cam=0.0)
    a, b = orc.Oracle(slow).trace(5.0, 2.0), orc.Oracle(fast).trace(5.0, 2.0)
    assert a["nsampled"] == b["nsampled"] > 50
    assert a["I"][0] == pytest.approx(b["I"][0], rel=1e-13) and a["I"][0] > 0


def test_flux_is_the_pixel_sum_in_jansky():
    s = scenes.config_C0(4)
    o = orc.Oracle(s)
    img = np.arange(16, dtype=float).reshape(1, 4, 4) * 1e-10
    L = 6.6743e-8 * s.M_bh_g / C_ ** 2
    expect = img.sum() * (s.fov_M / 4) ** 2 * L ** 2 / s.D_src_cm ** 2 * 1e23
    assert o.flux(img)[0] == pytest.approx(expect, rel=1e-13)


# ------------------------------------------------------------------------------------ P14
def _c1_flux(nx, refine=1.0):
    s = scenes.config_C1(nx)
    s = replace(s, step_c=s.step_c / refine, step_min=s.step_min / refine, step_max=s.step_max / refine,
                eps_polar=s.eps_polar / refine)
    o = orc.Oracle(s)
    out = o.render()
    return o.flux(out["image"])[0], out


def test_P14_whole_image_step_refinement_and_resolution_convergence():
    # (i) the geodesics are 4th order, the quadrature of Eq. 37 with one end-point sample per step [A8] is 1st
    # order: halving every step halves the flux error.  (iii) the total flux converges with the image resolution,
    # the differences between successive resolutions shrinking as in Table 3.
    f1, _ = _c1_flux(24, 1.0)
    f2, _ = _c1_flux(24, 2.0)
    f4, _ = _c1_flux(24, 4.0)
    assert abs(f1 - f2) / f4 < 0.05                       # the contract step rule is within a few % of converged
    assert 1.5 < (f1 - f2) / (f2 - f4) < 2.7, ((f1 - f2) / (f2 - f4))
    fr = [_c1_flux(n)[0] for n in (8, 16, 32, 64)]
    d = np.abs(np.diff(fr))
    assert d[2] < d[0] and d[2] / fr[-1] < 0.05, (fr, d)
    # every pixel's intensity is non-negative and the image is mirror-symmetric about beta = 0 only in flux
    # between the two halves for the equatorially symmetric torus seen from i = 60 deg: NOT symmetric (Doppler
    # boosting): the approaching side (alpha < 0, Eq. 25) is brighter
    _, out = _c1_flux(32)
    img = out["image"][0]
    assert (img >= 0).all() and img[:, :16].sum() > 1.2 * img[:, 16:].sum()


# --------------------------------------------------------------- optical-depth cut-off (Table 2 :335)
def test_tau_cutoff_exit_status_step_count_and_governing_frequency(golden):
    # Uniform static slab in flat space, constant step: tau grows by the same d_tau on every sampled step, so the
    # iteration at which "min_k tau_k > tau_cutoff" (O4: tested at the START of an iteration [A7]) first holds can
    # be counted by hand from the UNCUT ray: n_stop = (steps before the slab) + floor(cutoff/d_tau) + 1.
    cut = golden["tau_cutoff"]
    assert cut == pytest.approx(math.log(1000.0), rel=1e-15)
    hstep = 0.05

    def slab(freqs, tau_cutoff):
        return replace(scenes.slab_scene(2e8, 10.0, 30.0, 8.0, sin_pitch=1.0, step_c=0.0, step_min=hstep, step_max=hstep,
                                         eps_polar=1e30, r_cam=60.0, incl_deg=30.0), freq_hz=freqs, tau_cutoff=tau_cutoff)

    nu_a, nu_b = 230e9, 460e9
    free = orc.Oracle(slab((nu_a, nu_b), math.inf))
    ref = free.trace(4.0, 3.0, record_path=True)
    assert ref["status"] == 2
    z = np.exp(ref["path"][:, 1]) * np.cos(math.pi * ref["path"][:, 2])
    inside = np.abs(z) < 4.0
    first = int(np.argmax(inside))                  # 0-based index of the first sampled step = steps taken before it
    n_in = int(inside.sum())
    assert ref["nsampled"] == n_in and inside[first:first + n_in].all()
    dtau = ref["tau"] / n_in                        # per sampled step, per frequency (uniform medium, nu_hat = 1)
    assert dtau[0] > 2 * dtau[1] and n_in * dtau[1] > 2 * cut          # 460 GHz is the more transparent one
    # hand check of d_tau itself: alpha L h with Kirchhoff alpha = j/B_nu (both pinned above)
    for k, nu in enumerate((nu_a, nu_b)):
        alpha = orc.emissivity(nu, 2e8, 10.0, 30.0, 1.0) / orc.planck(nu, 10.0)
        assert dtau[k] == pytest.approx(alpha * free.scene.L_cm * hstep, rel=1e-12)
    # single frequency: stops right after tau first EXCEEDS the cut-off
    for k, nu in enumerate((nu_a, nu_b)):
        r = orc.Oracle(slab((nu,), cut)).trace(4.0, 3.0)
        m = int(math.floor(cut / dtau[k])) + 1      # sampled steps needed: m d_tau > cut >= (m-1) d_tau
        assert r["status"] == 4                     # THICK
        assert r["nsampled"] == m and r["nsteps"] == first + m, (r["nsteps"], first, m)
        assert r["tau"][0] == pytest.approx(m * dtau[k], rel=1e-12) and r["tau"][0] > cut >= r["tau"][0] - dtau[k]
        # the intensity is the formal solution up to that depth: nothing behind tau = ln 1000 is added
        assert r["I"][0] == pytest.approx(orc.planck(nu, 10.0) * (1 - math.exp(-m * dtau[k])), rel=1e-11)
    # two frequencies: the SMALLER optical depth governs (the ray goes on while any frequency can still see through)
    r2 = orc.Oracle(slab((nu_a, nu_b), cut)).trace(4.0, 3.0)
    m_b = int(math.floor(cut / dtau[1])) + 1
    assert r2["status"] == 4 and r2["nsampled"] == m_b and r2["nsteps"] == first + m_b
    assert r2["tau"][1] > cut and r2["tau"][0] > 2 * cut
    # a cut-off the slab never reaches changes nothing; cut-off 0 stops after the first sampled step (tau > 0)
    r3 = orc.Oracle(slab((nu_a, nu_b), 1e6)).trace(4.0, 3.0)
    assert r3["status"] == 2 and r3["nsteps"] == ref["nsteps"] and np.array_equal(r3["I"], ref["I"])
    r4 = orc.Oracle(slab((nu_a,), 0.0)).trace(4.0, 3.0)
    assert r4["status"] == 4 and r4["nsampled"] == 1 and r4["nsteps"] == first + 1
