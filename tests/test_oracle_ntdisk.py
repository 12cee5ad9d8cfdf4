"""Pins for the oracle's Novikov-Thorne disk (model kind 4, reading NT of eq. (35)).

The paper prints eq. (35), F = 3 Mdot M f / (8 pi r^3) = sigma T_eff^4, without f(r).  The oracle uses Page & Thorne's
closed form; here it is pinned against things that do not share its algebra:
  * the conservation-law integral it is the antiderivative of, done by quadrature on Bardeen's circular-orbit E, L, Omega;
  * energy conservation of the whole disk: the luminosity at infinity equals Mdot (1 - E_isco);
  * its Newtonian limit 1 - sqrt(r_isco / r);
  * the Newtonian temperature in cgs at large radius, typed with its own constants;
  * the observed intensity against the Planck law and its Rayleigh-Jeans and Wien limits;
  * a face-on spectrum against a direct radial quadrature.
"""
import math

import numpy as np
import pytest
from scipy import integrate

import workloads as W
from oracle import binding as O

G, C, H, KB, SIG = 6.67430e-8, 2.99792458e10, 6.62607015e-27, 1.380649e-16, 5.670374419e-5
GM_SUN = 1.3271244e26


def circ(a, r):
    """Bardeen, Press & Teukolsky (1972) prograde circular equatorial orbits: E, L, Omega (M = 1)."""
    d = math.sqrt(1.0 - 3.0 / r + 2.0 * a * r ** -1.5)
    E = (1.0 - 2.0 / r + a * r ** -1.5) / d
    L = math.sqrt(r) * (1.0 - 2.0 * a * r ** -1.5 + a * a / (r * r)) / d
    Om = 1.0 / (r ** 1.5 + a)
    return E, L, Om


def f_by_quadrature(a, r):
    """Page & Thorne (1974): F = Mdot/(4 pi r) * [-Omega_,r (E - Omega L)^-2 int_{r_ms}^{r} (E - Omega L) L_,r dr];
    eq. (35)'s f is that times 8 pi r^3 / (3 Mdot)."""
    r0 = O.kerr_constants(a)["r_isco"]

    def dLdr(s):
        h = 1e-5 * s
        return (circ(a, s + h)[1] - circ(a, s - h)[1]) / (2 * h)

    def integrand(s):
        E, L, Om = circ(a, s)
        return (E - Om * L) * dLdr(s)

    val, _ = integrate.quad(integrand, r0, r, epsabs=1e-13, epsrel=1e-12, limit=400)
    E, L, Om = circ(a, r)
    dOm = -1.5 * math.sqrt(r) / (r ** 1.5 + a) ** 2
    return (2.0 * r * r / 3.0) * (-dOm) * val / (E - Om * L) ** 2


@pytest.mark.parametrize("a", [0.0, 0.5, 0.9, 0.998])
def test_closed_form_equals_conservation_law_integral(a):
    r0 = O.kerr_constants(a)["r_isco"]
    for r in (1.05 * r0, 1.5 * r0, 3.0 * r0, 20.0, 300.0):
        assert O.page_thorne_f(a, r) == pytest.approx(f_by_quadrature(a, r), rel=2e-6, abs=1e-9)


@pytest.mark.parametrize("a", [0.0, 0.7, 0.998])
def test_disk_luminosity_is_the_binding_energy_at_the_isco(a):
    # energy conservation: int_{r_ms}^{inf} 4 pi r F E dr = Mdot (1 - E_ms); with eq. (35), F = 3 Mdot f / (8 pi r^3)
    r0 = O.kerr_constants(a)["r_isco"]
    val, _ = integrate.quad(lambda u: 1.5 * O.page_thorne_f(a, 1.0 / u) * circ(a, 1.0 / u)[0], 0.0, 1.0 / r0,
                            epsabs=1e-12, epsrel=1e-11, limit=400)      # u = 1/r: dr / r^2 = -du
    assert val == pytest.approx(1.0 - circ(a, r0)[0], rel=1e-7)
    if a == 0.0:
        assert val == pytest.approx(1.0 - math.sqrt(8.0 / 9.0), rel=1e-7)   # the textbook 5.72 %


def test_inner_edge_and_newtonian_limit():
    for a in (0.0, 0.9, 0.998):
        r0 = O.kerr_constants(a)["r_isco"]
        assert O.page_thorne_f(a, r0) == 0.0
        assert O.page_thorne_f(a, 0.9 * r0) == 0.0
        assert 0.0 < O.page_thorne_f(a, r0 * (1 + 1e-6)) < 1e-4
        fs = [O.page_thorne_f(a, r) for r in (1e3, 1e5, 1e7)]
        assert fs[0] < fs[1] < fs[2] < 1.0
        # the Newtonian factor carries the sqrt(r0/r); the relativistic remainder is O(ln r / sqrt r)
        for r in (1e5, 1e7):
            assert O.page_thorne_f(a, r) == pytest.approx(1.0 - math.sqrt(r0 / r), abs=0.5 * math.log(r) / math.sqrt(r))


def test_temperature_matches_the_newtonian_disk_in_cgs_far_out():
    mo = W.model_nt_disk(mbh_msun=10.0, mdot_gs=1e19)
    M = 10.0 * GM_SUN / G
    a = 0.3
    r0 = O.kerr_constants(a)["r_isco"]
    for r in (20.0, 1e4, 1e6):
        R = r * G * M / C ** 2                       # eq. (35) in cgs: sigma T^4 = 3 G M Mdot f / (8 pi R^3)
        T_newton = (3.0 * G * M * 1e19 * (1.0 - math.sqrt(r0 / r)) / (8.0 * math.pi * SIG * R ** 3)) ** 0.25
        T_quad = (3.0 * G * M * 1e19 * f_by_quadrature(a, r) / (8.0 * math.pi * SIG * R ** 3)) ** 0.25
        assert O.nt_temperature(mo, a, r) == pytest.approx(T_quad, rel=1e-6)
        if r > 100.0:
            assert O.nt_temperature(mo, a, r) == pytest.approx(T_newton, rel=0.2 * math.log(r) / math.sqrt(r))
    # T_eff^4 is linear in Mdot and, at fixed r in r_g, falls as M^-2
    t1 = O.nt_temperature(mo, a, 12.0)
    assert O.nt_temperature(W.model_nt_disk(10.0, 16e19), a, 12.0) == pytest.approx(2.0 * t1, rel=1e-13)
    assert O.nt_temperature(W.model_nt_disk(160.0, 1e19), a, 12.0) == pytest.approx(0.25 * t1, rel=1e-13)
    assert O.nt_temperature(mo, a, 0.5 * r0) == 0.0
    # Fig. 6's set-up (M = 10 M_sun, Mdot = 1e19 g/s): the inner disk is at ~1e7 K, i.e. kT ~ 1 keV
    assert 5e6 < O.nt_temperature(mo, 0.0, 10.0) < 2e7


def test_pixel_intensity_is_the_redshifted_planck_law():
    a, inc = 0.9, 60.0
    sc = W.scene(a, inc, 24, 18.0)
    mo = W.model_nt_disk(r_out=15.0)
    kev = 2.417989242e17
    nu = [1e-4 * kev, 0.3 * kev, 1.0 * kev, 30.0 * kev]
    sp = O.render_spectrum(sc, mo, nu)
    thin = dict(W.model_thin_disk(r_in=0.0, r_out=15.0))
    im = O.render_image(sc, thin, 0.0)
    g, re, flag = im["aux0"], im["aux1"], im["flag"]
    assert np.array_equal(flag, sp["flag"])                       # same geometry as the thin disk
    hit = flag == 2
    assert hit.sum() > 60
    for q, f in enumerate(nu):
        I = sp["images"][q]
        assert np.all(I[~hit] == 0.0)
        T = np.array([O.nt_temperature(mo, a, r) for r in re[hit]])
        x = H * f / (g[hit] * KB * T)
        planck = 2.0 * H * f ** 3 / C ** 2 / np.expm1(x)
        np.testing.assert_allclose(I[hit], planck, rtol=1e-12)
        if q == 0:      # Rayleigh-Jeans: I = 2 nu^2 k (g T) / c^2
            np.testing.assert_allclose(I[hit], 2.0 * f * f * KB * g[hit] * T / C ** 2, rtol=2e-3)
        if q == 3:      # Wien: ln I = ln(2 h nu^3 / c^2) - x
            sel = x > 20
            assert sel.sum() > 10
            np.testing.assert_allclose(np.log(I[hit][sel]), math.log(2.0 * H * f ** 3 / C ** 2) - x[sel], rtol=1e-9)
    # approaching side is blue-shifted and brighter at high frequency than the receding side at the same row
    row = sp["images"][2].reshape(24, 24)[12]
    assert row[:12].sum() != row[12:].sum()


def test_face_on_spectrum_matches_a_radial_quadrature():
    # i -> 0, a = 0, large disk: light bending moves the apparent radius by ~1 M and the redshift of a circular
    # orbit seen face-on is g = sqrt(1 - 3/r); nu L_nu = 4 pi nu r_g^2 int I_nu(r) 2 pi r dr
    a, r_out = 0.0, 1500.0
    mo = W.model_nt_disk(mbh_msun=10.0, mdot_gs=1e19, r_out=r_out)
    sc = W.scene(a, 0.5, 160, 1600.0)
    sc["r_obs"] = 1.0e5
    sc["r_esc"] = 1.1e5
    kev = 2.417989242e17
    nu = [1e-3 * kev, 1e-2 * kev, 0.05 * kev, 0.25 * kev]
    got = O.render_spectrum(sc, mo, nu)["nuLnu"]
    rg = 10.0 * GM_SUN / C ** 2
    for q, f in enumerate(nu[:3]):
        def integrand(r):
            T = O.nt_temperature(mo, a, r)
            gg = math.sqrt(1.0 - 3.0 / r)
            return 2.0 * H * f ** 3 / C ** 2 / math.expm1(H * f / (gg * KB * T)) * 2.0 * math.pi * r
        val, _ = integrate.quad(integrand, 6.0 + 1e-9, r_out, limit=400)
        assert got[q] == pytest.approx(4.0 * math.pi * f * rg * rg * val, rel=0.015)
    # Rayleigh-Jeans tail of the outer edge (nu L_nu ~ nu^3) below k T(r_out) ~ 10 eV, and the multi-temperature
    # nu L_nu ~ nu^(4/3) between k T(r_out) and k T_max ~ 1 keV
    assert 2.8 < math.log(got[1] / got[0]) / math.log(10.0) < 3.0
    assert 1.0 < math.log(got[3] / got[2]) / math.log(5.0) < 1.5
