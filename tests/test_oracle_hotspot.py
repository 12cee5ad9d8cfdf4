"""Pins for the oracle's hot-spot model (kind 3; reading HS of PAPER.md:L252-264, eq. (36), Figs. 7, 8): a
Gaussian spot co-rotating on the opaque equatorial plane, seen at the emission time t_obs + t_e."""
import math

import numpy as np
import pytest
from scipy import special

import workloads as W
from oracle import binding as O


def _period(a, rs):
    return 2.0 * math.pi * (rs ** 1.5 + a)


def test_pixel_values_follow_eq36_at_the_retarded_spot_position():
    """Rebuild every pixel of every phase from the ray's own (g, r_e, phi_e, t_e): wiring of the model."""
    a, rs, sig, phi0, p = 0.5, 7.0, 0.8, 0.3, 4.0
    sc = W.scene(a, 55.0, 48, 11.0)
    mo = W.model_hot_spot(r_orbit=rs, r_spot=sig, phi0=phi0, g_power=p)
    t_obs = np.array([0.0, 11.0, 57.5, 140.0])
    o = O.render_hotspot(sc, mo, t_obs)
    hit = o["flag"] == W.FLAG_DISK
    assert hit.sum() > 500 and np.all(o["t_e"][hit] < -900.0) and np.all(o["t_e"][~hit] == 0.0)
    Om = 1.0 / (rs ** 1.5 + a)
    Re, Rs = np.sqrt(o["r_e"] ** 2 + a * a), math.sqrt(rs * rs + a * a)
    for k, t in enumerate(t_obs):
        phis = phi0 + Om * (t + o["t_e"])
        d2 = Re ** 2 + Rs ** 2 - 2 * Re * Rs * np.cos(o["phi_e"] - phis)
        want = np.where(hit & (d2 < 16 * sig * sig), o["g"] ** p * np.exp(-d2 / (2 * sig * sig)), 0.0)
        assert np.allclose(o["images"][k], want, rtol=1e-12, atol=0.0)
        assert (o["images"][k] > 0).sum() > 3
    area = (22.0 / 48) ** 2
    assert np.allclose(o["lightcurve"], o["images"].sum(axis=1) * area, rtol=1e-13)
    # spectrogram: flux of each phase binned over g
    assert np.allclose(o["spectrogram"].sum(axis=1), o["lightcurve"], rtol=1e-12)


def test_geometry_of_the_crossing_is_the_thin_disk_one():
    sc = W.scene(0.9, 60.0, 40, 12.0)
    hs = O.render_hotspot(sc, W.model_hot_spot(), [0.0])
    # the hot-spot plane reaches inwards to the inner edge of the spot: R_in = sqrt(r_s^2 + a^2) - 4 r_spot (reading HS)
    kc = O.kerr_constants(0.9)
    R_in = math.sqrt(kc["r_isco"] ** 2 + 0.81) - 4 * 0.5
    assert R_in < 0.9                                              # here the inner edge lies inside the hole: the plane is lit down to the capture radius
    td = O.render_image(sc, W.model_thin_disk(r_in=1e-9))
    assert np.array_equal(hs["flag"], td["flag"])
    assert np.array_equal(hs["g"], td["aux0"]) and np.array_equal(hs["r_e"], td["aux1"])


def test_light_curve_is_periodic_with_the_orbital_period():
    a, rs = 0.3, 6.5
    sc = W.scene(a, 70.0, 40, 10.0)
    mo = W.model_hot_spot(r_orbit=rs, r_spot=1.0)
    T = _period(a, rs)
    t = np.array([13.0, 40.0, 77.0])
    f0 = O.render_hotspot(sc, mo, t)["lightcurve"]
    f1 = O.render_hotspot(sc, mo, t + T)["lightcurve"]
    f3 = O.render_hotspot(sc, mo, t - 3 * T)["lightcurve"]
    assert np.all(f0 > 0)
    assert np.allclose(f1, f0, rtol=1e-9) and np.allclose(f3, f0, rtol=1e-8)


def test_face_on_light_curve_is_flat():
    """Seen along the spin axis the system is axisymmetric: moving the spot round its orbit only rotates the
    image, so the flux does not depend on the phase (up to the pixel sampling of a rotating pattern)."""
    a, rs = 0.0, 8.0
    sc = W.scene(a, 0.01, 160, 14.0)                     # the field holds the whole spot (8 + 4 x 1.0 < 14) at every phase
    mo = W.model_hot_spot(r_orbit=rs, r_spot=1.0)
    t = np.linspace(0.0, _period(a, rs), 9)[:-1]
    f = O.render_hotspot(sc, mo, t)["lightcurve"]
    assert f.min() > 0 and (f.max() - f.min()) / f.mean() < 5e-3
    # edge-on the same spot is strongly modulated (beaming + lensing)
    f85 = O.render_hotspot(W.scene(a, 85.0, 96, 14.0), mo, t)["lightcurve"]
    assert f85.max() / f85.min() > 5.0


def test_phase_average_equals_bessel_closed_form():
    """Average of exp(-d^2/2s^2) over one orbit at fixed (R_e, phi_e) is exp(-(R_e^2+R_s^2)/2s^2) I_0(R_e R_s/s^2)
    (the 4 r_spot cut removes < 4e-4 of it); it does not depend on phi_e or t_e.  With 32 equally spaced phases the
    periodic trapezoid rule is exact to ~1e-9 for R_e R_s / s^2 ~ 16."""
    a, rs, sig = 0.0, 6.0, 1.5
    sc = W.scene(a, 40.0, 40, 11.0)
    mo = W.model_hot_spot(r_orbit=rs, r_spot=sig, g_power=3.0)
    t = np.linspace(0.0, _period(a, rs), 33)[:-1]
    o = O.render_hotspot(sc, mo, t)
    avg = o["images"].mean(axis=0)
    hit = (o["flag"] == W.FLAG_DISK) & (np.abs(o["r_e"] - rs) < 2.0)
    Re = o["r_e"][hit]
    want = o["g"][hit] ** 3.0 * np.exp(-(Re ** 2 + rs ** 2) / (2 * sig * sig)) * special.i0(Re * rs / sig ** 2)
    assert hit.sum() > 50
    assert np.allclose(avg[hit], want, rtol=3e-3)


def test_flux_peaks_when_the_approaching_spot_is_seen():
    """Edge-on, the brightest phase is the one whose emission-time position is on the approaching (blue) side:
    the flux-weighted g at the peak of the light curve exceeds 1 and exceeds the one at the minimum."""
    a, rs = 0.0, 6.0
    sc = W.scene(a, 75.0, 64, 10.0)
    mo = W.model_hot_spot(r_orbit=rs, r_spot=0.8)
    t = np.linspace(0.0, _period(a, rs), 25)[:-1]
    o = O.render_hotspot(sc, mo, t)
    kmax, kmin = int(np.argmax(o["lightcurve"])), int(np.argmin(o["lightcurve"]))
    gw = lambda k: (o["images"][k] * o["g"]).sum() / o["images"][k].sum()
    assert gw(kmax) > 1.0 > gw(kmin)


def test_lit_region_is_the_whole_gaussian_symmetric_about_the_orbit():
    """everything within d < 4 r_spot of the centre is lit, and the centre orbits AT r_isco — so the lit
    region must extend as far inside the orbit as outside it (with the thin disk's inner edge r_isco as the plane's
    edge the inner half of the spot would be dark).  Seen nearly face-on, a = 0: lit crossings span r_s - 2 .. r_s + 2."""
    sc = W.scene(0.0, 0.5, 160, 10.0)
    mo = W.model_hot_spot(r_spot=0.5)
    out = O.render_hotspot(sc, mo, [0.0])
    lit = out["images"][0] > 0
    assert lit.sum() > 100
    re = out["r_e"][lit]
    assert re.min() == pytest.approx(6.0 - 2.0, abs=0.15) and re.max() == pytest.approx(6.0 + 2.0, abs=0.15)
    # and the brightest pixel sits at the centre of the spot, not at the plane's edge
    assert out["r_e"][np.argmax(out["images"][0])] == pytest.approx(6.0, abs=0.15)
