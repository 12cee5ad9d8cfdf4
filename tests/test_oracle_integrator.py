"""Pins for the oracle's Runge-Kutta pairs, controller and invariants (CPU only).

Cites: PAPER.md:L90 (fifth-order RK with adaptive step, Press et al. 1992); L50, eq. (13) (constants of
motion); SURVEY.md §8(c) rows "Integrator", "Invariants", reading R.
"""
import math

import numpy as np
import pytest

import workloads as W
from oracle import binding as O


def _order_conditions(c, A, b, order):
    """Rooted-tree order conditions up to `order` (Butcher); returns list of (lhs, rhs)."""
    Ac = A @ c
    conds = [(b.sum(), 1.0)]
    if order >= 2:
        conds += [(b @ c, 1 / 2)]
    if order >= 3:
        conds += [(b @ c ** 2, 1 / 3), (b @ Ac, 1 / 6)]
    if order >= 4:
        conds += [(b @ c ** 3, 1 / 4), (b @ (c * Ac), 1 / 8), (b @ (A @ c ** 2), 1 / 12), (b @ (A @ Ac), 1 / 24)]
    if order >= 5:
        conds += [(b @ c ** 4, 1 / 5), (b @ (c ** 2 * Ac), 1 / 10), (b @ (c * (A @ c ** 2)), 1 / 15),
                  (b @ (c * (A @ Ac)), 1 / 30), (b @ (Ac * Ac), 1 / 20), (b @ (A @ c ** 3), 1 / 20),
                  (b @ (A @ (c * Ac)), 1 / 40), (b @ (A @ (A @ c ** 2)), 1 / 60), (b @ (A @ (A @ Ac)), 1 / 120)]
    return conds


@pytest.mark.parametrize("which", [W.TABLEAU_RKF45, W.TABLEAU_CASH_KARP])
def test_tableau_order_conditions(which):
    c, A, b5, b4 = O.tableau(which)
    assert np.allclose(A.sum(axis=1), c, atol=1e-15)            # row sums
    assert np.all(np.triu(A) == 0.0)                            # explicit
    for lhs, rhs in _order_conditions(c, A, b5, 5):
        assert lhs == pytest.approx(rhs, abs=2e-16)
    for lhs, rhs in _order_conditions(c, A, b4, 4):
        assert lhs == pytest.approx(rhs, abs=2e-16)
    # the embedded solution is NOT fifth order (otherwise the error estimate would vanish)
    assert max(abs(l - r) for l, r in _order_conditions(c, A, b4, 5)) > 1e-4


def test_rkf45_first_row_is_fehlberg():
    """Spot values every textbook prints for Fehlberg's pair."""
    c, A, b5, b4 = O.tableau(W.TABLEAU_RKF45)
    assert c[3] == 12 / 13 and A[3, 1] == -7200 / 2197 and b5[3] == 28561 / 56430 and b4[2] == 1408 / 2565


@pytest.mark.parametrize("which", [W.TABLEAU_RKF45, W.TABLEAU_CASH_KARP])
def test_observed_order_is_five(which):
    """Fixed-step integration over a strongly curved stretch of a Kerr geodesic: the error of the
    propagated (5th-order) solution falls by ~2^5 per halving, the embedded estimate by ~2^5 per step
    (local error O(h^5) of the 4th-order companion)."""
    a = 0.9
    sc = W.scene(a, 60.0, 64, 10.0)
    st, cons = O.init_ray(sc, 4.0, 3.0)
    # bring the ray close to the hole with the adaptive driver, then take fixed steps from r ~ 12
    nodes, cons2, _ = O.trace_path(dict(sc, rtol=1e-12), W.model_none(), 4.0, 3.0)
    k = int(np.argmax(nodes[:, 0] < 12.0))
    y0 = nodes[k]
    span = 6.0

    def run(n):
        y = y0.copy()
        h = span / n
        for _ in range(n):
            y, _ = O.rk_attempt(a, cons["E"], cons["L"], which, y, h)
        return y

    ref = run(4096)
    errs = [np.max(np.abs(run(n) - ref)) for n in (16, 32, 64)]
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(4.6 < o < 5.6 for o in orders), (errs, orders)
    # embedded error estimate scales as h^5
    e1 = np.max(np.abs(O.rk_attempt(a, cons["E"], cons["L"], which, y0, 0.4)[1]))
    e2 = np.max(np.abs(O.rk_attempt(a, cons["E"], cons["L"], which, y0, 0.2)[1]))
    assert 4.5 < math.log2(e1 / e2) < 5.6


def test_error_norm_scaling():
    """err = max_i |e_i| / sc_i / rtol with sc = (|r|, 1, 1, 1+|p_r|, 1+|p_theta|) (reading G)."""
    y = np.array([50.0, 1.0, 2.0, -3.0, 0.5])
    assert O.error_norm(y, [5e-7, 0, 0, 0, 0], 1e-8) == pytest.approx(1.0)
    assert O.error_norm(y, [0, 2e-8, 0, 0, 0], 1e-8) == pytest.approx(2.0)
    assert O.error_norm(y, [0, 0, -3e-8, 0, 0], 1e-8) == pytest.approx(3.0)
    assert O.error_norm(y, [0, 0, 0, 4e-8, 0], 1e-8) == pytest.approx(1.0)
    assert O.error_norm(y, [0, 0, 0, 0, 3e-8], 1e-8) == pytest.approx(2.0)
    assert math.isnan(O.error_norm(y, [float("nan"), 0, 0, 0, 0], 1e-8))


@pytest.mark.parametrize("a,incl,rtol,bound_esc,bound_cap", [
    (0.0, 60.0, 1e-8, 1e-7, 1e-6), (0.9, 60.0, 1e-10, 5e-9, 5e-8), (0.998, 85.0, 1e-12, 1e-10, 1e-9)])
def test_null_condition_and_carter_constant_along_rays(a, incl, rtol, bound_esc, bound_cap):
    """Along every accepted node the scale-free null ratio (reading R) and Q (eq. (13)) stay at the
    level the tolerance allows.  north_star's '|dH| < 1e-10 at tolerance 1e-10' is read this way."""
    sc = W.scene(a, incl, 64, 10.0, rtol=rtol)
    worst = {0: 0.0, 1: 0.0}
    worstQ = 0.0
    for (x, y) in [(-9.0, 1.0), (-4.0, 3.0), (0.5, 0.5), (2.0, -1.0), (5.5, 0.3), (8.0, -7.0), (-1.0, 5.3)]:
        nodes, cons, res = O.trace_path(sc, W.model_none(), x, y)
        assert res["flag"] in (W.FLAG_ESCAPED, W.FLAG_CAPTURED)
        ratios = [abs(O.null_ratio(a, cons["E"], cons["L"], n)) for n in nodes]
        worst[res["flag"]] = max(worst[res["flag"]], max(ratios))
        Qs = np.array([O.carter_Q(a, cons["E"], cons["L"], n) for n in nodes])
        worstQ = max(worstQ, np.max(np.abs(Qs - cons["Q"])) / (1.0 + abs(cons["Q"])))
    assert worst[0] < bound_esc and worst[1] < bound_cap, worst
    assert worstQ < 50 * max(bound_esc, bound_cap)


def test_step_controller_accept_reject_statistics():
    """Attempt/accept counters: every ray needs far fewer than max_attempts, rejections are a minority,
    and tightening rtol by 100 multiplies the accepted steps by about 100^(1/5) (5th-order method)."""
    pts = [(-6.0, 2.0), (3.0, 4.0), (7.0, -1.0)]
    xs, ys = zip(*pts)
    lo = O.trace_points(W.scene(0.9, 60.0, 64, 10.0, rtol=1e-8), W.model_none(), [], xs, ys)
    hi = O.trace_points(W.scene(0.9, 60.0, 64, 10.0, rtol=1e-10), W.model_none(), [], xs, ys)
    assert np.all(lo["n_attempt"] < 1000) and np.all(lo["n_accept"] <= lo["n_attempt"])
    assert np.all(lo["n_attempt"] - lo["n_accept"] < 0.5 * lo["n_attempt"])
    ratio = hi["n_accept"].sum() / lo["n_accept"].sum()
    assert 1.8 < ratio < 3.2, ratio          # 100^(1/5) = 2.51


def test_step_sequence_is_that_of_press_et_als_controller():
    """PAPER.md:L90 cites Press et al. (1992) for the step control; their driver (rkqs) uses SAFETY 0.9, PGROW -0.2,
    PSHRNK -0.25, ERRCON 1.89e-4 (growth at most x 5) and shrinks by at most x 10 (reading G).  The oracle's accepted
    step lengths are re-derived here from those numbers, with the oracle's embedded pair and error norm as black boxes:
    starting from h0, every trial step is accepted iff err <= 1, h <- h min(5, 0.9 err^-0.2) after an accepted step and
    h <- h max(0.1, 0.9 err^-0.25) after a rejected one.  Swapping the two exponents, or another safety factor,
    changes the sequence at its first rejection and fails the comparison (checked for the swap below)."""
    sc = W.scene(0.9, 60.0, 64, 10.0, rtol=1e-8)
    a = sc["a"]
    for x, y in [(-6.0, 2.0), (7.0, -1.0)]:
        nodes, cons, res = O.trace_path(sc, W.model_none(), x, y)
        st, _ = O.init_ray(sc, x, y)
        h_acc = np.diff(nodes[:, 5])                                    # accepted step lengths (node 0 is the start; the last step is event-located)

        def simulate(pgrow, pshrnk, n_steps):
            yv, h, out, attempts = np.array(st[:5], float), sc["h0"], [], 0
            while len(out) < n_steps:
                ynew, yerr = O.rk_attempt(a, cons["E"], cons["L"], sc["tableau"], yv, h)
                err = O.error_norm(yv, yerr, sc["rtol"])
                attempts += 1
                if err <= 1.0:
                    out.append(h); yv = ynew
                    h *= 5.0 if err < 1.89e-4 else min(5.0, 0.9 * err ** pgrow)
                else:
                    h *= max(0.1, 0.9 * err ** pshrnk)
            return np.array(out), attempts
        n = len(h_acc) - 1                                              # all but the located last step
        sim, attempts = simulate(-0.2, -0.25, n)
        assert res["n_attempt"] > res["n_accept"]                       # the ray does have rejected attempts
        assert np.allclose(sim, h_acc[:n], rtol=1e-12, atol=0.0)
        swapped, _ = simulate(-0.25, -0.2, n)
        assert not np.allclose(swapped, h_acc[:n], rtol=1e-6, atol=0.0)
