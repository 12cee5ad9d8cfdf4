"""Pins for the oracle's traced geodesics against what general relativity fixes (CPU only).

Cites: PAPER.md:L215-219 (shadow; alpha^2 + beta^2 = 27; analytic Kerr solution); L50 (constants of
motion); SURVEY.md §8(c) rows "Capture classification", "Shadow edge", "Deflection", reading S.
"""
import math

import mpmath
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import kerr_reference as K
import workloads as W
from oracle import binding as O


def _bisect_edge(sc, p_in, p_out, tol=1e-10):
    """Bisect along the image-plane segment p_in (captured) -> p_out (escaping)."""
    p_in, p_out = np.array(p_in, float), np.array(p_out, float)
    f = lambda p: O.trace_points(sc, W.model_none(), [], [p[0]], [p[1]])["flag"][0]
    assert f(p_in) == W.FLAG_CAPTURED and f(p_out) == W.FLAG_ESCAPED
    while np.linalg.norm(p_out - p_in) > tol:
        mid = 0.5 * (p_in + p_out)
        if f(mid) == W.FLAG_CAPTURED:
            p_in = mid
        else:
            p_out = mid
    return 0.5 * (p_in + p_out)


@pytest.mark.parametrize("angle_deg", [0.0, 37.0, 90.0, 200.0])
def test_schwarzschild_shadow_radius_is_sqrt27(angle_deg):
    """for a = 0 the shadow follows alpha^2 + beta^2 = 27.  The edge ray's impact parameter
    b = sqrt(L^2 + Q) (E = 1) must be 3 sqrt(3); in pixel units from r_obs = 1000 that is
    sqrt(27) (1 - 27/r_obs^3 ...) = 5.19615228 (finite-distance shift of eqs. (7),(8))."""
    sc = W.scene(0.0, 60.0, 64, 10.0, rtol=1e-10)
    u = np.array([math.cos(math.radians(angle_deg)), math.sin(math.radians(angle_deg))])
    edge = _bisect_edge(sc, 4.0 * u, 6.5 * u)
    _, cons = O.init_ray(sc, edge[0], edge[1])
    b = math.sqrt(cons["L"] ** 2 + cons["Q"])
    assert b == pytest.approx(math.sqrt(27.0), abs=2e-7)
    assert np.linalg.norm(edge) == pytest.approx(5.1961522824, abs=5e-7)


@pytest.mark.parametrize("a", [0.5, 0.9, 0.9375, 0.998])
def test_kerr_equatorial_shadow_edges_are_bardeen_critical_impact_parameters(a):
    """Observer in the equatorial plane, beta = 0: the shadow's edges are the critical impact parameters
    of the prograde / retrograde circular photon orbits, alpha = -xi(r_ph)  (Bardeen 1973; the "analytic
    solution" drawn in the paper's Fig. 4).  Prograde edge on the LEFT (reading B)."""
    sc = W.scene(a, 90.0, 64, 10.0, rtol=1e-10)
    r_pro, r_ret = K.photon_orbit_radii(a)
    xi_pro, _ = K.critical_xi_eta(a, r_pro)
    xi_ret, _ = K.critical_xi_eta(a, r_ret)
    assert xi_pro > 0 > xi_ret
    left = _bisect_edge(sc, (0.5, 0.0), (-9.0, 0.0))
    right = _bisect_edge(sc, (0.5, 0.0), (9.0, 0.0))
    # image coordinate = -xi up to the O(a/r_obs) finite-distance shift of eq. (8) (the 2arE term: about
    # 2a/r_obs = 2e-3 a); the conserved lambda of the edge ray, below, is the sharp statement
    assert left[0] == pytest.approx(-xi_pro, abs=3e-3)
    assert right[0] == pytest.approx(-xi_ret, abs=3e-3)
    for edge, xi in ((left, xi_pro), (right, xi_ret)):
        _, cons = O.init_ray(sc, edge[0], 0.0)
        assert -cons["L"] == pytest.approx(xi, abs=3e-7)       # lambda_phys = -L (k-type)
        assert abs(cons["Q"]) < 1e-20


def test_closed_form_values_of_survey_table():
    """SURVEY.md §8(c) 'Values': r_h, r_isco, r_ph, xi for a = 0.9 (closed forms; Bardeen, Press & Teukolsky)."""
    k = O.kerr_constants(0.9)
    assert k["r_h"] == pytest.approx(1.43588989, abs=1e-8)
    assert k["r_isco"] == pytest.approx(2.32088304, abs=1e-8)
    r_pro, r_ret = K.photon_orbit_radii(0.9)
    assert (r_pro, r_ret) == pytest.approx((1.55785463, 3.91026794), abs=1e-8)
    assert O.kerr_constants(0.0)["r_isco"] == pytest.approx(6.0, abs=1e-14)
    assert O.kerr_constants(0.0)["E_isco"] == pytest.approx(math.sqrt(8.0 / 9.0), abs=1e-15)
    assert O.kerr_constants(0.0)["L_isco"] == pytest.approx(math.sqrt(12.0), abs=1e-14)
    assert O.kerr_constants(-0.9)["r_isco"] == pytest.approx(8.71735, abs=1e-5)      # retrograde ISCO, a = 0.9


@pytest.mark.parametrize("a,incl", [(0.0, 60.0), (0.5, 45.0), (0.9, 60.0), (0.9375, 30.0), (0.998, 85.0), (-0.9, 70.0)])
def test_capture_classification_every_pixel_equals_closed_form(a, incl):
    """Every pixel of a 48x48 image: captured iff R(r) = (r^2+a^2-a lam)^2 - Delta[(lam-a)^2+q] has no real
    root outside the horizon (lam = L_phys/E_phys = -L, q = Q).  Independent of any integrator."""
    sc = W.scene(a, incl, 48, 10.0)
    out = O.trace_geodesics(sc)
    flags = out["flag"].reshape(48, 48)
    assert set(np.unique(flags)) <= {W.FLAG_ESCAPED, W.FLAG_CAPTURED}
    dx = 20.0 / 48
    n_cap = 0
    for j in range(48):
        for i in range(48):
            x, y = -10.0 + (i + 0.5) * dx, -10.0 + (j + 0.5) * dx
            _, cons = O.init_ray(sc, x, y)
            want = K.captured_closed_form(a, -cons["L"], cons["Q"])
            assert (flags[j, i] == W.FLAG_CAPTURED) == want, (i, j)
            n_cap += want
    assert 100 < n_cap < 1200


def test_final_state_lies_on_the_stopping_surface():
    sc = W.scene(0.9, 60.0, 32, 10.0)
    out = O.trace_geodesics(sc)
    rh = K.horizon(0.9)
    esc = out["flag"] == W.FLAG_ESCAPED
    assert np.max(np.abs(out["r"][esc] - sc["r_esc"])) < 1e-9
    assert np.max(np.abs(out["r"][~esc] - (rh + sc["horizon_eps"]))) < 1e-12
    assert np.all(out["n_accept"] <= out["n_attempt"])


@pytest.mark.parametrize("b0", [6.0, 8.0, 20.0, 150.0])
def test_schwarzschild_deflection_equals_orbit_integral(b0):
    """a = 0, equatorial: total swept azimuth between the start radius and r_esc equals the textbook orbit
    integral  dphi = int dr / (r^2 sqrt(1/b^2 - (1 - 2/r)/r^2))  evaluated by tanh-sinh quadrature."""
    sc = W.scene(0.0, 90.0, 64, 10.0, rtol=1e-11)
    st, cons = O.init_ray(sc, b0, 0.0)
    b = abs(cons["L"])
    out = O.trace_points(sc, W.model_none(), [], [b0], [0.0])
    assert out["flag"][0] == W.FLAG_ESCAPED
    swept = abs(out["ph"][0] - st[2])
    with mpmath.workdps(30):
        # f(u) = 1/b^2 - u^2 (1 - 2u) = 2 (u - u1)(u2 - u)(u3 - u), u = 1/r; periastron u2 = smallest positive
        # root; the substitution u = u2 - s^2 removes the square-root singularity there.
        roots = sorted(mpmath.polyroots([2, -1, 0, 1 / mpmath.mpf(b) ** 2], maxsteps=200, extraprec=200),
                       key=lambda z: z.real)
        u1, u2, u3 = [z.real for z in roots]
        assert u1 < 0 < u2 < u3
        integ = lambda u0: mpmath.quad(lambda t: 2 / mpmath.sqrt(2 * (u2 - t * t - u1) * (u3 - u2 + t * t)),
                                       [0, mpmath.sqrt(u2 - u0)])
        want = float(integ(1 / mpmath.mpf(st[0])) + integ(1 / mpmath.mpf(out["r"][0])))
    assert swept == pytest.approx(want, abs=2e-9)
    if b0 >= 150.0:   # weak-field limit 4/b + 15 pi/(4 b^2) for the part beyond pi (finite end radii subtracted)
        straight = math.pi - math.asin(b / st[0]) - math.asin(b / out["r"][0])
        assert swept - straight == pytest.approx(4 / b + 15 * math.pi / (4 * b * b), rel=2e-2)


@pytest.mark.parametrize("a,incl,x,y", [(0.9, 60.0, -5.0, 3.0), (0.998, 85.0, 7.5, 0.5), (0.5, 30.0, 2.0, -6.5)])
def test_against_independent_8_component_hamiltonian_integration(a, incl, x, y):
    """The same ray integrated as an 8-component (x^mu, p_mu) Hamiltonian system with scipy's DOP853 on
    Hamilton's equations derived symbolically from eq. (1): there p_t and p_phi are integrated (their
    drift is the E, L_z conservation of north_star) and nothing of the oracle's RHS or stepper is used."""
    sc = W.scene(a, incl, 64, 10.0, rtol=1e-11)
    st, cons = O.init_ray(sc, x, y)
    out = O.trace_points(sc, W.model_none(), [], [x], [y])
    assert out["flag"][0] == W.FLAG_ESCAPED

    def f(lam, s):
        t, r, th, ph, pt, pr, pth, pph = s
        d = K.hamilton_rhs(a, r, th, pt, pr, pth, pph)
        return [d[0], d[1], d[2], d[3], 0.0, d[4], d[5], 0.0]   # dH/dt = dH/dphi = 0 exactly (Killing)

    def reached(lam, s):
        return s[1] - sc["r_esc"] if s[5] > 0 else -1.0
    reached.terminal, reached.direction = True, 1.0
    s0 = [0.0, st[0], st[1], st[2], -cons["E"], st[3], st[4], cons["L"]]
    sol = solve_ivp(f, [0.0, 5000.0], s0, method="DOP853", rtol=1e-12, atol=1e-14, events=reached)
    assert sol.status == 1
    end = sol.y_events[0][0]
    assert end[4] == -cons["E"] and end[7] == cons["L"]
    assert K.hamilton_rhs(a, end[1], end[2], end[4], end[5], end[6], end[7])[6] == pytest.approx(0.0, abs=1e-10)
    assert out["th"][0] == pytest.approx(end[2], abs=2e-8)
    assert out["ph"][0] == pytest.approx(end[3], abs=2e-8)


# ---- coordinate time, eq. (9) (the sixth of the six parameters of PAPER.md:L88) -------------------------
@pytest.mark.parametrize("a,incl,x,y", [(0.9, 60.0, -5.0, 3.0), (0.998, 85.0, 7.5, 0.5), (0.5, 30.0, 2.0, -6.5)])
def test_coordinate_time_against_independent_8_component_integration(a, incl, x, y):
    """t integrated with eq. (9) along the ray equals t of the independent Hamiltonian integration (dt/dlambda =
    dH/dp_t there).  E = -1: the ray is traced backwards, so t runs to negative values."""
    sc = W.scene(a, incl, 64, 10.0, rtol=1e-11)
    st, cons = O.init_ray(sc, x, y)
    out = O.trace_points(sc, W.model_none(), [], [x], [y])

    def f(lam, s):
        t, r, th, ph, pt, pr, pth, pph = s
        d = K.hamilton_rhs(a, r, th, pt, pr, pth, pph)
        return [d[0], d[1], d[2], d[3], 0.0, d[4], d[5], 0.0]

    def reached(lam, s):
        return s[1] - sc["r_esc"] if s[5] > 0 else -1.0
    reached.terminal, reached.direction = True, 1.0
    s0 = [0.0, st[0], st[1], st[2], -cons["E"], st[3], st[4], cons["L"]]
    sol = solve_ivp(f, [0.0, 5000.0], s0, method="DOP853", rtol=1e-12, atol=1e-14, events=reached)
    end = sol.y_events[0][0]
    assert out["t"][0] < -1900.0
    assert out["t"][0] == pytest.approx(end[0], abs=2e-7)


def test_eq9_slope_equals_hamilton_equation_for_t():
    rng = np.random.default_rng(3)
    for _ in range(40):
        a = rng.uniform(-0.99, 0.99); r = rng.uniform(2.2, 40.0); th = rng.uniform(0.2, 2.9)
        L = rng.uniform(-6, 6); pr = rng.uniform(-1, 1); pth = rng.uniform(-4, 4)
        dy = O.rhs(a, -1.0, L, [r, th, 0.0, pr, pth], with_t=True)
        d = K.hamilton_rhs(a, r, th, 1.0, pr, pth, L)       # p_t = -E = +1
        assert dy[5] == pytest.approx(d[0], rel=1e-12)


@pytest.mark.parametrize("b0", [6.0, 20.0, 150.0])
def test_schwarzschild_travel_time_equals_orbit_integral(b0):
    """a = 0, equatorial: elapsed coordinate time between the start radius and r_esc equals the textbook
    integral  dt = dr / ((1 - 2/r) sqrt(1 - b^2 (1 - 2/r)/r^2))  (two legs, tanh-sinh quadrature); for large b
    it is the straight-line time plus the first-order (Shapiro) delay
    2 ln[(r1 + sqrt(r1^2 - r0^2))(r2 + sqrt(r2^2 - r0^2))/r0^2] + sqrt((r1 - r0)/(r1 + r0)) + sqrt((r2 - r0)/(r2 + r0)),
    r0 the periastron."""
    sc = W.scene(0.0, 90.0, 64, 10.0, rtol=1e-11)
    st, cons = O.init_ray(sc, b0, 0.0)
    b = abs(cons["L"])
    out = O.trace_points(sc, W.model_none(), [], [b0], [0.0])
    assert out["flag"][0] == W.FLAG_ESCAPED
    with mpmath.workdps(30):
        bb = mpmath.mpf(b)
        rp = max(z.real for z in mpmath.polyroots([1, 0, -bb ** 2, 2 * bb ** 2], maxsteps=200, extraprec=200))
        # r = rp + s^2 removes the inverse-square-root singularity at the periastron
        def leg(r_end):
            g = lambda s: 2 * s / ((1 - 2 / (rp + s * s)) * mpmath.sqrt(abs(1 - bb ** 2 * (1 - 2 / (rp + s * s)) / (rp + s * s) ** 2)))
            return mpmath.quad(g, [0, mpmath.sqrt(mpmath.mpf(r_end) - rp)])
        want = float(leg(st[0]) + leg(out["r"][0]))
    assert -out["t"][0] == pytest.approx(want, rel=1e-9)
    if b0 >= 150.0:
        r1, r2, r0 = st[0], out["r"][0], float(rp)            # Weinberg's first-order formula is in the periastron r0
        s1, s2 = math.sqrt(r1 * r1 - r0 * r0), math.sqrt(r2 * r2 - r0 * r0)
        straight = s1 + s2
        shapiro = 2.0 * math.log((r1 + s1) * (r2 + s2) / (r0 * r0)) + math.sqrt((r1 - r0) / (r1 + r0)) + math.sqrt((r2 - r0) / (r2 + r0))
        assert -out["t"][0] - straight == pytest.approx(shapiro, rel=2e-2)


def test_conditioning_of_rays_of_a_nearly_polar_observer():
    """What the GPU parity test's allowance for observers 0.1 degrees from the axis rests on: there the problem itself
    amplifies a one-ulp change of the image coordinate (a relative perturbation of 1e-16) to more than 1e-9 of the
    end state — a condition number above 1e7 — while for an observer at 60 degrees the same perturbation moves
    nothing by more than 1e-10.  Oracle only."""
    def worst_move(a, incl):
        sc = W.scene(a, incl, 48, 12.0, ny=40)
        dx, dy = (sc["x_max"] - sc["x_min"]) / sc["nx"], (sc["y_max"] - sc["y_min"]) / sc["ny"]
        xs = np.array([sc["x_min"] + (i + 0.5) * dx for j in range(sc["ny"]) for i in range(sc["nx"])])
        ys = np.array([sc["y_min"] + (j + 0.5) * dy for j in range(sc["ny"]) for i in range(sc["nx"])])
        o0 = O.trace_points(sc, W.model_none(), [], list(xs), list(ys))
        o1 = O.trace_points(sc, W.model_none(), [], list(np.nextafter(xs, np.inf)), list(ys))
        assert np.array_equal(o0["flag"], o1["flag"])
        return max(np.max(np.abs(o0[k] - o1[k]) / np.maximum(np.abs(o0[k]), 1.0)) for k in ("r", "th", "ph"))
    assert worst_move(0.9999, 0.1) > 1e-9
    assert worst_move(0.9, 60.0) < 1e-10
