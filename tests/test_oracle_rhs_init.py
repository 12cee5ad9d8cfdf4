"""Pins for the oracle's right-hand side and initial conditions (CPU only).

Cites: eq. (1); L52-64 eqs. (3)-(8); L68-88 eqs. (9)-(15); L94-102 eqs. (16),(17);
L104-143 eqs. (18)-(26).  SURVEY.md §8(c) rows "RHS" and "Init".
"""
import math

import numpy as np
import pytest

import workloads as W
from oracle import binding as O
import kerr_reference as K

RNG = np.random.default_rng(20160121)


def _random_point(on_shell):
    a = RNG.uniform(-0.998, 0.998)
    rh = K.horizon(a)
    r = rh + 10 ** RNG.uniform(-1.0, 1.7)
    th = RNG.uniform(0.05, math.pi - 0.05)
    L = RNG.uniform(-8.0, 8.0)
    pth = RNG.uniform(-6.0, 6.0)
    E = -1.0
    if on_shell:
        Delta = r * r - 2 * r + a * a
        P = (r * r + a * a) * E - a * L
        D = L / math.sin(th) - a * E * math.sin(th)
        pr2 = (P * P / Delta - pth * pth - D * D) / Delta
        if pr2 < 0:
            return _random_point(on_shell)
        pr = math.copysign(math.sqrt(pr2), RNG.uniform(-1, 1))
    else:
        pr = RNG.uniform(-2.0, 2.0)
    return a, E, L, np.array([r, th, RNG.uniform(-3, 3), pr, pth])


@pytest.mark.parametrize("on_shell", [True, False])
def test_rhs_equals_hamilton_equations_of_eq1(on_shell):
    """rdot..pthdot equal dH/dp, -dH/dx of H = 1/2 g^{mu nu} p_mu p_nu with g from eq. (1), derived
    symbolically and evaluated in 40-digit arithmetic.  Off-shell points test the G terms of reading A."""
    worst = 0.0
    for _ in range(60):
        a, E, L, y = _random_point(on_shell)
        ref = K.hamilton_rhs(a, y[0], y[1], -E, y[3], y[4], L, high_precision=True)
        got = O.rhs(a, E, L, y)
        want = np.array([ref[1], ref[2], ref[3], ref[4], ref[5]])
        scale = np.maximum(np.abs(want), 1e-3 * np.max(np.abs(want)))
        worst = max(worst, np.max(np.abs(got - want) / scale))
    assert worst < 5e-12


def test_rhs_reduces_to_printed_eqs_14_15_on_shell():
    """On the null shell the Hamiltonian form equals eqs. (14),(15) as printed (mu = 0)."""
    worst = 0.0
    for _ in range(200):
        a, E, L, y = _random_point(True)
        r, th, _, pr, pth = y
        s, c = math.sin(th), math.cos(th)
        Sigma = r * r + a * a * c * c
        Delta = r * r - 2 * r + a * a
        kappa = pth ** 2 + L ** 2 / s ** 2 + a * a * E * E * s * s                        # L88 with mu = 0
        pr_dot = (-kappa * (r - 1.0) + 2.0 * r * (r * r + a * a) * E * E - 2.0 * a * E * L) / (Sigma * Delta) \
            - 2.0 * pr * pr * (r - 1.0) / Sigma                                          # eq. (14), mu = 0
        pth_dot = s * c / Sigma * (L * L / s ** 4 - a * a * E * E)                       # eq. (15), mu = 0
        got = O.rhs(a, E, L, y)
        worst = max(worst, abs(got[3] - pr_dot) / (abs(pr_dot) + 1e-3), abs(got[4] - pth_dot) / (abs(pth_dot) + 1e-3))
    assert worst < 1e-9       # limited by the on-shell p_r solved in double precision


def test_phidot_is_eq12_and_rdot_thdot_are_eqs_4_5():
    for _ in range(50):
        a, E, L, y = _random_point(False)
        r, th, _, pr, pth = y
        s, c = math.sin(th), math.cos(th)
        Sigma = r * r + a * a * c * c
        Delta = r * r - 2 * r + a * a
        got = O.rhs(a, E, L, y)
        assert got[0] == pytest.approx(Delta * pr / Sigma, rel=1e-14)                                  # eq. (4)
        assert got[1] == pytest.approx(pth / Sigma, rel=1e-14)                                         # eq. (5)
        assert got[2] == pytest.approx((2 * a * r * E + (Sigma - 2 * r) * L / s ** 2) / (Sigma * Delta), rel=1e-13)  # (12)


def test_pole_clamp():
    """sin(theta) is replaced by +-1e-8 when |sin theta| < 1e-8: finite RHS at the pole."""
    dy = O.rhs(0.9, -1.0, 1e-3, [5.0, 0.0, 0.0, -0.5, 0.3])
    assert np.all(np.isfinite(dy))
    dy_m = O.rhs(0.9, -1.0, 1e-3, [5.0, -1e-12, 0.0, -0.5, 0.3])
    assert np.all(np.isfinite(dy_m))
    assert dy_m[4] * dy[4] <= 0 or abs(dy[4]) == 0      # the clamp keeps the sign of sin(theta)


@pytest.mark.parametrize("a,incl", [(0.0, 60.0), (0.9, 60.0), (0.9375, 30.0), (0.998, 85.0), (-0.7, 120.0)])
def test_initial_state_is_null_and_matches_eqs_16_17(a, incl):
    sc = W.scene(a, incl, 64, 10.0)
    to = sc["theta_obs"]
    for (x, y) in [(3.0, 2.0), (-7.5, 0.4), (0.3, -9.0), (-2.0, -2.0)]:
        st, cons = O.init_ray(sc, x, y)
        E, L, Q = cons["E"], cons["L"], cons["Q"]
        assert E == -1.0
        assert abs(O.null_ratio(a, E, L, st)) < 5e-16
        # against the independent Hamiltonian: H = 0 with p_t = -E
        H = K.hamilton_rhs(a, st[0], st[1], -E, st[3], st[4], L, high_precision=True)[6]
        assert abs(H) < 1e-15
        # eqs. (16), (17) and "beta is also equal to the initial value of -p_theta" are
        # statements at r_obs = infinity: check them for the integrated (k-type) constants from 1e6 M.
        far = dict(sc, r_obs=1.0e6, r_esc=1.0e6)
        stf, cf = O.init_ray(far, x, y)
        alpha = cf["L"] / math.sin(to)
        beta2 = cf["Q"] + a * a * math.cos(to) ** 2 - cf["L"] ** 2 / math.tan(to) ** 2
        assert alpha == pytest.approx(x, abs=2e-4)
        assert math.sqrt(beta2) == pytest.approx(abs(y), abs=2e-4)
        assert -stf[4] == pytest.approx(y, abs=2e-4)
        # and from 1000 M they already hold to O(1/r_obs)
        assert L / math.sin(to) == pytest.approx(x, abs=0.02)
        # the ray starts inward
        assert st[3] < 0
        assert O.carter_Q(a, E, L, st) == pytest.approx(Q, rel=1e-14, abs=1e-14)


def test_schwarzschild_equatorial_closed_form_start():
    """a = 0, observer in the equatorial plane, y = 0: before the |E| normalisation L_z = r sin(Phi) = x
    exactly and E^2 = 1 - (2/r) sin^2(Phi)   (from eqs. (7),(8),(18)-(26) by hand)."""
    sc = W.scene(0.0, 90.0, 64, 10.0)
    for x in (-9.0, -3.3, 0.7, 5.2):
        st, cons = O.init_ray(sc, x, 0.0)
        r, th, ph = st[0], st[1], st[2]
        assert th == pytest.approx(math.pi / 2, abs=1e-15)
        assert r == pytest.approx(math.hypot(sc["r_obs"], x), rel=1e-15)
        assert cons["L_raw"] == pytest.approx(x, rel=1e-13)
        assert cons["E2_raw"] == pytest.approx(1.0 - (2.0 / r) * math.sin(ph) ** 2, rel=1e-14)
        assert st[4] == pytest.approx(0.0, abs=1e-13)


def test_pixel_to_position_matches_eq18_geometry():
    """Position from eqs. (18)-(22): for a = 0 the start point is at Euclidean distance
    sqrt(r_obs^2 + x^2 + y^2) and the image-plane offsets are orthogonal to the line of sight."""
    sc = W.scene(0.0, 60.0, 64, 10.0)
    to = sc["theta_obs"]
    n_los = np.array([math.sin(to), 0.0, math.cos(to)])       # from hole to observer (phi_obs = 0)
    for (x, y) in [(3.0, 2.0), (-7.5, 0.4)]:
        st, _ = O.init_ray(sc, x, y)
        r, th, ph = st[:3]
        pos = r * np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
        assert r == pytest.approx(math.sqrt(sc["r_obs"] ** 2 + x * x + y * y), rel=1e-14)
        assert pos @ n_los == pytest.approx(sc["r_obs"], rel=1e-14)
        # x is along +y' (observer's right for phi_obs = 0), y along the projected spin axis
        assert pos[1] == pytest.approx(x, abs=1e-12)
        e_up = np.array([-math.cos(to), 0.0, math.sin(to)])
        assert pos @ e_up == pytest.approx(y, abs=1e-12)
