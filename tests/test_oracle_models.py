"""Pins for the oracle's emission models and radiative-transfer update (CPU only).

Cites: eq. (2); L223, L244 (thin disk, Fig. 5); L149-171 eqs. (27)-(31);
L268-282 eqs. (37)-(39); SURVEY.md §8(c) rows "Thin-disk g", "RT".
"""
import math

import numpy as np
import pytest
from scipy import integrate, special

import kerr_reference as K
import workloads as W
from oracle import binding as O

RNG = np.random.default_rng(1601)


def _keplerian_g_closed_form(a, r, lam):
    """Cunningham 1975 (cited PAPER.md:L268): g = sqrt(1 - 3/r + 2a r^-3/2) / (1 + (a - lam) r^-3/2)."""
    return math.sqrt(1.0 - 3.0 / r + 2.0 * a * r ** -1.5) / (1.0 + (a - lam) * r ** -1.5)


def test_equatorial_keplerian_gamma_is_closed_form():
    """eq. (2) evaluated with the metric-built four-velocity equals the closed form; p_r, p_theta do not
    enter because u^r = u^theta = 0."""
    for _ in range(100):
        a = RNG.uniform(-0.99, 0.998)
        r = O.kerr_constants(a)["r_isco"] * (1.0 + 10 ** RNG.uniform(-3, 1.3))
        L = RNG.uniform(-6, 6)
        ok, u, g = O.flow_gamma(a, r, math.pi / 2, RNG.uniform(-1, 1), RNG.uniform(-3, 3), L)
        assert ok
        assert g == pytest.approx(_keplerian_g_closed_form(a, r, -L), rel=2e-14)
        # four-velocity is normalised: g_{mu nu} u^mu u^nu = -1 with the metric of eq. (1)
        gm = K.metric_cov(a, r, math.pi / 2)
        assert u @ gm @ u == pytest.approx(-1.0, abs=1e-12)


def test_flow_velocity_normalised_everywhere_and_plunging_inside_isco():
    """Keplerian shells off the equator and the plunging branch inside the ISCO (reading N):
    u.u = -1 with eq. (1)'s metric, u^r < 0 only inside r_isco, continuous across r_isco, and on the
    equator the plunging u has the ISCO's conserved u_t = -E_isco, u_phi = L_isco."""
    for a in (0.0, 0.5, 0.9375, 0.998):
        kc = O.kerr_constants(a)
        for r in np.linspace(kc["r_h"] + 0.02, 12.0, 25):
            for th in (0.2, 1.0, math.pi / 2, 2.3):
                ok, u, _ = O.flow_gamma(a, r, th, 0.0, 0.0, 0.0)
                assert ok
                gm = K.metric_cov(a, r, th)
                assert u @ gm @ u == pytest.approx(-1.0, abs=1e-10)
                assert (u[1] < 0) == (r < kc["r_isco"]) or abs(u[1]) < 1e-7
                assert u[2] == 0.0 and u[0] > 0
        r = 0.5 * (kc["r_h"] + kc["r_isco"])
        _, u, _ = O.flow_gamma(a, r, math.pi / 2, 0.0, 0.0, 0.0)
        u_cov = K.metric_cov(a, r, math.pi / 2) @ u
        assert -u_cov[0] == pytest.approx(kc["E_isco"], rel=1e-12)
        assert u_cov[3] == pytest.approx(kc["L_isco"], rel=1e-12)
        eps = 1e-9
        _, u_in, _ = O.flow_gamma(a, kc["r_isco"] - eps, 1.1, 0.0, 0.0, 0.0)
        _, u_out, _ = O.flow_gamma(a, kc["r_isco"] + eps, 1.1, 0.0, 0.0, 0.0)
        assert np.allclose(u_in, u_out, atol=1e-6)


def test_fig5_thin_disk_orientation_and_range():
    """Fig. 5 set-up: a = 0, cos(theta_obs) = 0.25, disk r_isco..50.  'The approaching
    (left) side is blue shifted', contour levels run 0.55..1.3, radial contours 6.1..50.  The located
    crossing satisfies the closed form g(r_e, lambda) of the emitting orbit."""
    sc = W.scene(0.0, math.degrees(math.acos(0.25)), 64, 60.0, rtol=1e-10)
    md = W.model_thin_disk()
    out = O.render_image(sc, md)
    g = out["aux0"].reshape(64, 64)
    hit = out["flag"].reshape(64, 64) == W.FLAG_DISK
    assert hit.sum() > 500
    left, right = g[:, :32][hit[:, :32]], g[:, 32:][hit[:, 32:]]
    assert left.mean() > 1.0 > right.mean()
    assert 1.3 < g[hit].max() < 1.4 and 0.45 < g[hit].min() < 0.55
    re = out["aux1"][out["flag"] == W.FLAG_DISK]
    assert re.min() >= 6.0 and re.max() <= 50.0
    pts = O.trace_points(sc, md, [], [-10.0, 10.0], [0.0, 0.0])
    assert list(pts["flag"]) == [W.FLAG_DISK, W.FLAG_DISK]
    for k, x in enumerate((-10.0, 10.0)):
        _, cons = O.init_ray(sc, x, 0.0)
        assert pts["g"][k] == pytest.approx(_keplerian_g_closed_form(0.0, pts["r_e"][k], -cons["L"]), rel=1e-13)
        assert abs(pts["th"][k] - math.pi / 2) < 1e-12
    assert pts["g"][0] == pytest.approx(1.26907, abs=2e-5) and pts["g"][1] == pytest.approx(0.60304, abs=2e-5)
    assert pts["r_e"][1] == pytest.approx(9.04791, abs=2e-5)
    # image value and line-profile histogram (BASELINE.json:configs[1])
    val = out["image"][out["flag"] == W.FLAG_DISK]
    gg = out["aux0"][out["flag"] == W.FLAG_DISK]
    assert np.allclose(val, gg ** 3 * re ** -3.0, rtol=1e-13)
    area = (120.0 / 64) ** 2
    assert out["hist"].sum() == pytest.approx(val.sum() * area, rel=1e-12)
    b = np.floor(gg / 2.0 * 200).astype(int)
    assert np.allclose(out["hist"], np.bincount(b, weights=val * area, minlength=200), rtol=1e-12, atol=0)


def test_disk_is_opaque_first_crossing_wins_and_gap_rays_pass_through():
    """Reading P: a ray that crosses the equatorial plane inside [r_in, r_out] stops there; one that crosses
    inside the inner edge goes on (captured or escaping)."""
    sc = W.scene(0.9, 60.0, 64, 70.0)
    out = O.render_image(sc, W.model_thin_disk())
    fl = out["flag"].reshape(64, 64)
    assert {W.FLAG_DISK, W.FLAG_CAPTURED, W.FLAG_ESCAPED} == set(np.unique(fl))
    kc = O.kerr_constants(0.9)
    re = out["aux1"][out["flag"] == W.FLAG_DISK]
    assert re.min() >= kc["r_isco"] and re.max() <= 50.0


def test_K2_matches_scipy():
    for x in np.logspace(math.log10(0.02), math.log10(60.0), 60):
        assert O.bessel_K2(x) == pytest.approx(special.kv(2, x), rel=5e-14)


def test_mahadevan_fit_value_printed_in_eq38():
    """eq. (38) at x_M = 1: 4.0505 (1 + 0.40 + 0.5316) exp(-1.8899)."""
    assert O.mahadevan_M(1.0) == pytest.approx(4.0505 * 1.9316 * math.exp(-1.8899), rel=1e-15)
    # exponents: x^-1/6 prefactor, x^-1/4 and x^-1/2 corrections, exp(-1.8899 x^1/3)
    x = 64.0
    want = 4.0505 / 2.0 * (1 + 0.40 / 64 ** 0.25 + 0.5316 / 8.0) * math.exp(-1.8899 * 4.0)
    assert O.mahadevan_M(x) == pytest.approx(want, rel=1e-14)


@pytest.mark.parametrize("xM", [0.3, 3.0, 30.0, 300.0])
def test_mahadevan_fit_approximates_the_thermal_synchrotron_integral(xM):
    """M(x_M) of eq. (38) is Mahadevan, Narayan & Yi (1996)'s fit to the angle-averaged ultra-relativistic
    thermal synchrotron integral I'(x_M) = (1/4pi) int I(x_M / sin t) dOmega,
    I(x) = (1/x) int_0^inf z^2 e^-z F(x / z^2) dz,  F(y) = y int_y^inf K_5/3.  The fit is good to a few per cent:
    this pins coefficients, exponents and the overall factor of the oracle's M()."""
    def F(y):
        return y * integrate.quad(lambda t: special.kv(5.0 / 3.0, t), y, np.inf, limit=200)[0]

    def I(x):
        return integrate.quad(lambda z: z * z * math.exp(-z) * F(x / (z * z)), 0.0, np.inf, limit=200)[0] / x

    Ip = integrate.quad(lambda t: 0.5 * math.sin(t) * I(xM / math.sin(t)), 1e-6, math.pi - 1e-6, limit=100)[0]
    assert O.mahadevan_M(xM) == pytest.approx(Ip, rel=0.06)


def test_planck_function_limits():
    nu, T = 1.0e9, 1.0e10
    k_B, c, h = 1.380649e-16, 2.99792458e10, 6.62607015e-27
    assert O.planck_B(nu, T) == pytest.approx(2 * nu * nu * k_B * T / c ** 2, rel=1e-6)         # Rayleigh-Jeans
    nu = 1e15; T = 5e3
    assert O.planck_B(nu, T) == pytest.approx(2 * h * nu ** 3 / c ** 2 * math.exp(-h * nu / (k_B * T)), rel=1e-3)  # Wien
    # Stefan-Boltzmann: pi int B_nu dnu = sigma T^4
    T = 1.0e4
    tot = integrate.quad(lambda x: O.planck_B(x * k_B * T / h, T), 1e-6, 60.0)[0] * k_B * T / h
    assert math.pi * tot == pytest.approx(5.670374419e-5 * T ** 4, rel=1e-6)


def test_plasma_profile_of_config2():
    """BASELINE.json:configs[2]: n_e = 1e7 (r/r_h)^-1.1 exp(-z^2 / 2(0.3 r)^2), T_e = 1e11 (r/r_h)^-0.84, B from beta = 10."""
    md = W.model_riaf()
    a = 0.9375
    rh = K.horizon(a)
    s = O.synchrotron(md, a, rh, math.pi / 2, 230e9)
    assert s["n_e"] == pytest.approx(1e7, rel=1e-14) and s["T_e"] == pytest.approx(1e11, rel=1e-14)
    s2 = O.synchrotron(md, a, 10 * rh, math.pi / 2, 230e9)
    assert s2["n_e"] == pytest.approx(1e7 * 10 ** -1.1, rel=1e-13)
    assert s2["T_e"] == pytest.approx(1e11 * 10 ** -0.84, rel=1e-13)
    s3 = O.synchrotron(md, a, 10 * rh, math.pi / 3, 230e9)            # z = r cos(theta)
    assert s3["n_e"] / s2["n_e"] == pytest.approx(math.exp(-0.25 / (2 * 0.09)), rel=1e-13)
    # magnetisation: P_gas / P_mag = beta with P_gas = n m_p c^2 / (6 r)  (reading O); B ~ 68 G at the horizon
    m_p, c = 1.67262192369e-24, 2.99792458e10
    assert (s["n_e"] * m_p * c * c / (6 * rh)) / (s["B"] ** 2 / (8 * math.pi)) == pytest.approx(10.0, rel=1e-13)
    assert 60 < s["B"] < 75
    assert s["Theta_e"] == pytest.approx(1.380649e-16 * 1e11 / (9.1093837015e-28 * c * c), rel=1e-14)
    # eq. (39): nu_c = 3 e B Theta^2 / (4 pi m_e c) = 1.5 nu_gyro Theta^2, nu_gyro = 2.799e6 B Hz
    assert s["nu_c"] == pytest.approx(1.5 * 2.7992e6 * s["B"] * s["Theta_e"] ** 2, rel=1e-4)
    # Kirchhoff
    assert s["alpha"] == pytest.approx(s["j"] / O.planck_B(230e9, s["T_e"]), rel=1e-14)
    # j is linear in n_e at fixed B, T: doubling j_scale doubles j
    sj = O.synchrotron(dict(md, j_scale=2.0), a, rh, math.pi / 2, 230e9)
    assert sj["j"] == pytest.approx(2 * s["j"], rel=1e-15)


def test_synchrotron_emissivity_ultrarelativistic_limit():
    """eq. (37) per steradian (reading F) in the limit Theta >> 1 where K_2(1/Theta) -> 2 Theta^2:
    j = n e^2 nu M(x_M) / (2 sqrt(3) c Theta^2)."""
    md = W.model_riaf(T0=1e13)
    a = 0.0
    s = O.synchrotron(md, a, 2.0, math.pi / 2, 1e12)
    e, c = 4.80320471257e-10, 2.99792458e10
    want = s["n_e"] * e * e * 1e12 * O.mahadevan_M(1e12 / s["nu_c"]) / (2 * math.sqrt(3) * c * s["Theta_e"] ** 2)
    assert s["j"] == pytest.approx(want, rel=1e-5)
    assert O.rg_cm(4.0e6) == pytest.approx(5.9068e11, rel=1e-4)        # G M / c^2 for 4e6 M_sun


def test_rt_update_uniform_slab_is_exact():
    """Constant coefficients, arbitrary step sizes: I = S (1 - exp(-tau)) exactly (formal solution, eq. (28))."""
    a_c, e_c = 0.37, 2.5e-3
    tau, T, I = 0.0, 1.0, 0.0
    lam = 0.0
    for dl in RNG.uniform(0.01, 3.0, size=40):
        tau, T, I = O.rt_update(a_c, a_c, e_c, e_c, dl, 1e30, tau, T, I)
        lam += dl
        assert tau == pytest.approx(a_c * lam, rel=1e-13)
        assert T == pytest.approx(math.exp(-tau), rel=1e-12)
        assert I == pytest.approx(e_c / a_c * (1 - math.exp(-tau)), rel=1e-12)


def test_rt_update_limits_and_freeze():
    # optically thin: plain trapezoid of eq. (31)
    tau, T, I = O.rt_update(0.0, 0.0, 1.0, 3.0, 0.5, 30.0, 0.0, 1.0, 0.0)
    assert (tau, T, I) == (0.0, 1.0, 1.0)
    # very thick single step: I -> S, no overflow
    tau, T, I = O.rt_update(1e6, 1e6, 2e6, 2e6, 1.0, 1e30, 0.0, 1.0, 0.0)
    assert I == pytest.approx(2.0, rel=1e-12) and T == 0.0
    # attenuation by material in front: contribution scaled by T = exp(-tau)
    _, _, I2 = O.rt_update(0.0, 0.0, 1.0, 1.0, 1.0, 30.0, 2.0, math.exp(-2.0), 0.0)
    assert I2 == pytest.approx(math.exp(-2.0), rel=1e-15)
    # frozen once tau > tau_max
    assert O.rt_update(1.0, 1.0, 1.0, 1.0, 1.0, 30.0, 30.5, 1e-14, 7.0) == (30.5, 1e-14, 7.0)


def test_rt_along_ray_optically_thin_limit_equals_independent_quadrature():
    """With a tiny density the image is the optically thin integral of eq. (31), int eps dlambda, along the ray.
    Rebuild eps at the accepted nodes from the public pieces (flow_gamma, synchrotron, rg_cm) and integrate
    (a) by the trapezoid rule over the same nodes: equals the driver's accumulated intensity to round-off
    (wiring: coefficient caching, step length of truncated steps, region limits); (b) over the nodes of a
    much finer path with Simpson-grade accuracy: equals it to the trapezoid truncation level."""
    a, nu = 0.9375, 230e9
    sc = W.scene(a, 30.0, 64, 15.0, rtol=1e-9)
    md = W.model_riaf(n0=1e2)
    x, y = 4.0, -3.0
    rg = O.rg_cm(md["mbh_msun"])
    rh = K.horizon(a)

    def thin_integral(rtol):
        nodes, cons, _ = O.trace_path(dict(sc, rtol=rtol), W.model_none(), x, y)
        eps = []
        for n in nodes:
            if not (rh + sc["horizon_eps"] < n[0] < md["r_rt_out"]):
                eps.append(0.0)
                continue
            ok, u, gam = O.flow_gamma(a, n[0], n[1], n[3], n[4], cons["L"])
            assert ok and gam > 0
            s = O.synchrotron(md, a, n[0], n[1], nu / gam)
            eps.append(rg * s["j"] / (gam * (nu / gam) ** 3))
        eps, lam = np.array(eps), nodes[:, 5]
        return float(np.sum(0.5 * (eps[1:] + eps[:-1]) * np.diff(lam)))

    out = O.trace_points(sc, md, [nu], [x], [y])
    assert 0 < out["tau"][0, 0] < 1e-6
    assert out["I"][0, 0] == pytest.approx(thin_integral(1e-9), rel=1e-11)
    assert out["I"][0, 0] == pytest.approx(thin_integral(1e-13), rel=5e-3)


def test_rt_along_ray_with_absorption_equals_formal_solution_on_a_fine_path():
    """Full transfer (emission AND absorption) along one ray: the driver's intensity must equal the formal
    solution of eqs. (30), (31),  I = int eps(l) exp(-tau(l)) dl,  tau(l) = int_0^l a dl',  evaluated
    independently (cumulative trapezoid for tau, trapezoid for I) on a MUCH finer path (rtol 1e-13: ~8x
    more nodes).  The driver's exact-attenuation update and the plain quadrature share only the public
    coefficient pieces; they agree to the truncation level of the coarse path.  nu = 30 GHz: tau ~ O(1-10)."""
    a, nu = 0.9375, 30e9
    sc = W.scene(a, 30.0, 64, 15.0, rtol=1e-9)
    md = W.model_riaf()
    x, y = 5.0, 2.0
    rg = O.rg_cm(md["mbh_msun"])
    rh = K.horizon(a)
    nodes, cons, _ = O.trace_path(dict(sc, rtol=1e-13), W.model_none(), x, y)
    eps, ab = [], []
    for n in nodes:
        if not (rh + sc["horizon_eps"] < n[0] < md["r_rt_out"]):
            eps.append(0.0); ab.append(0.0)
            continue
        ok, u, gam = O.flow_gamma(a, n[0], n[1], n[3], n[4], cons["L"])
        assert ok and gam > 0
        s = O.synchrotron(md, a, n[0], n[1], nu / gam)
        eps.append(rg * s["j"] / (gam * (nu / gam) ** 3))
        ab.append(rg * s["alpha"] / gam)
    eps, ab, lam = np.array(eps), np.array(ab), nodes[:, 5]
    dl = np.diff(lam)
    tau = np.concatenate([[0.0], np.cumsum(0.5 * (ab[1:] + ab[:-1]) * dl)])
    f = eps * np.exp(-tau)
    I_formal = float(np.sum(0.5 * (f[1:] + f[:-1]) * dl))
    out = O.trace_points(sc, md, [nu], [x], [y])
    assert 0.5 < out["tau"][0, 0] < 30.0                      # genuinely absorbing, not frozen
    assert out["tau"][0, 0] == pytest.approx(tau[-1], rel=2e-3)
    assert out["I"][0, 0] == pytest.approx(I_formal, rel=5e-3)


def test_riaf_image_converges_under_rtol_refinement():
    """The RIAF image as a whole has no value printed in the paper (its end-to-end pin is
    tests/test_oracle_riaf_independent.py); here: it converges as the step tolerance is refined."""
    w = W.C2(n=20)
    imgs = []
    for rtol in (1e-6, 1e-8, 1e-10):
        sc = dict(w["scene"], rtol=rtol)
        imgs.append(O.render_image(sc, w["model"], w["nu"][0])["image"])
    d1 = np.abs(imgs[0] - imgs[2]).sum() / imgs[2].sum()
    d2 = np.abs(imgs[1] - imgs[2]).sum() / imgs[2].sum()
    assert d2 < d1 < 0.05
    assert d2 < 5e-3


# ---- reading E': tau and I as Runge-Kutta components (workloads.RT_RK_COMPONENTS) ---------------------
@pytest.mark.parametrize("which", [W.TABLEAU_RKF45, W.TABLEAU_CASH_KARP])
def test_rt_rk_step_constant_coefficients_closed_form_and_order(which):
    """Constant a, eps over a step: tau grows linearly (exact), I = eps e^-tau0 (1 - e^-(a h))/a up to the
    fifth-order quadrature error, which falls by ~2^6 per halving of h (local error O(h^6))."""
    c, _, _, _ = O.tableau(which)
    a, eps, tau0, I0 = 0.7, 3.0, 0.4, 1.25
    errs = []
    for h in (0.8, 0.4, 0.2):
        tau, I = O.rt_rk_step(which, [a] * 6, [eps] * 6, h, 30.0, tau0, I0)
        assert tau == pytest.approx(tau0 + a * h, rel=1e-15)
        exact = I0 + eps * math.exp(-tau0) * (1.0 - math.exp(-a * h)) / a
        errs.append(abs(I - exact))
    assert errs[0] < 5e-6
    assert 40 < errs[0] / errs[1] < 100 and 40 < errs[1] / errs[2] < 100
    # stage abscissae enter through the stage values of tau: a linear-in-lambda absorption a(l) = a0 + s l
    s, h = 0.5, 0.3
    tau, _ = O.rt_rk_step(which, [a + s * ci * h for ci in c], [0.0] * 6, h, 30.0, 0.0, 0.0)
    assert tau == pytest.approx(a * h + 0.5 * s * h * h, rel=1e-14)
    # frozen once tau > tau_max
    assert O.rt_rk_step(which, [1.0] * 6, [1.0] * 6, 1.0, 30.0, 30.5, 7.0) == (30.5, 7.0)


def test_rk_component_scheme_along_a_ray_equals_formal_solution():
    """Same ray and frequency as the per-step pin above; the Runge-Kutta-component scheme is of higher
    order in the step, so it sits closer to the fine-path formal solution than the per-step scheme."""
    a, nu = 0.9375, 30e9
    sc = W.scene(a, 30.0, 64, 15.0, rtol=1e-9)
    x, y = 5.0, 2.0
    I0 = O.trace_points(sc, W.model_riaf(), [nu], [x], [y])
    I1 = O.trace_points(sc, W.model_riaf(rt_scheme=W.RT_RK_COMPONENTS), [nu], [x], [y])
    fine = O.trace_points(dict(sc, rtol=1e-13), W.model_riaf(rt_scheme=W.RT_RK_COMPONENTS), [nu], [x], [y])
    assert I1["n_attempt"][0] == I0["n_attempt"][0]                # the geodesic alone controls the steps
    assert I1["tau"][0, 0] == pytest.approx(fine["tau"][0, 0], rel=1e-5)
    assert I1["I"][0, 0] == pytest.approx(fine["I"][0, 0], rel=1e-4)
    assert abs(I1["I"][0, 0] - fine["I"][0, 0]) < abs(I0["I"][0, 0] - fine["I"][0, 0])
    assert I0["I"][0, 0] == pytest.approx(fine["I"][0, 0], rel=5e-3)


def test_the_two_transfer_schemes_converge_to_the_same_image():
    """Cross-pin for the RIAF image as a whole (no printed value exists): two different discretisations
    of eqs. (30), (31) along identical geodesics approach each other as the tolerance is refined."""
    w = W.C2(n=16)
    d = []
    for rtol in (1e-6, 1e-8, 1e-10):
        sc = dict(w["scene"], rtol=rtol)
        a = O.render_image(sc, w["model"], w["nu"][0])
        b = O.render_image(sc, dict(w["model"], rt_scheme=W.RT_RK_COMPONENTS), w["nu"][0])
        assert np.array_equal(a["flag"], b["flag"]) and np.array_equal(a["n_attempt"], b["n_attempt"])
        d.append(np.abs(a["image"] - b["image"]).sum() / a["image"].sum())
    assert d[0] > d[1] > d[2]
    assert d[2] < 2e-4


# ------------------------------------------------------------------------------------------------
# Rays through the rotation axis (L_z = 0: the centre column of an image with an odd number of columns) continue
# with theta outside [0, pi]; they meet the equatorial plane at theta = pi/2 + k pi, the point (pi/2, phi + k pi).
# Pin: continuity with their neighbours at x = +/- 1e-3, whose L_z != 0 keeps them inside (0, pi).
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("a, incl", [(0.0, 120.0), (0.0, 60.0), (0.9, 100.0), (0.998, 175.0)])
def test_disk_crossing_of_rays_through_the_axis_is_continuous_with_their_neighbours(a, incl):
    sc = W.scene(a, incl, 3, 12.0)
    sc.update(ny=25, x_min=-1.5e-3, x_max=1.5e-3, y_min=-30.0, y_max=30.0)
    mo = W.model_hot_spot(r_spot=1.0)
    mo.update(r_in=0.0, r_out=60.0)
    out = O.render_hotspot(sc, mo, [0.0])
    flag = out["flag"].reshape(25, 3)
    assert flag.max() <= 2                                      # nobody stuck (MAXSTEP) on the axis
    r_e, g, phi = (out[k].reshape(25, 3) for k in ("r_e", "g", "phi_e"))
    rows = np.nonzero((flag == 2).all(axis=1))[0]
    assert len(rows) >= 12
    through_axis = 0
    for j in rows:
        if abs(r_e[j, 0] - r_e[j, 2]) > 0.5:                    # a row where the two neighbours see different image orders
            continue
        assert r_e[j, 1] == pytest.approx(0.5 * (r_e[j, 0] + r_e[j, 2]), abs=2e-4)
        assert g[j, 1] == pytest.approx(0.5 * (g[j, 0] + g[j, 2]), abs=2e-4)
        # azimuth of the crossing point, modulo 2 pi: the neighbours swing round the axis by +pi and -pi
        for k in (0, 2):
            assert np.cos(phi[j, 1] - phi[j, k]) == pytest.approx(1.0, abs=1e-3)
        through_axis += 1
    assert through_axis >= 10
