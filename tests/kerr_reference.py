"""Independent reference objects for pinning the oracle (test helper; not part of the oracle, not
part of the product).

Everything here is derived by computer algebra (sympy) or numerical linear algebra (numpy) directly
from the covariant Kerr metric printed as eq. (1) of the paper — NOT from the
oracle's formulas — so that a dropped term, wrong sign or transposed index in the oracle's
right-hand side fails the comparison.
"""
import functools

import numpy as np
import sympy as sp


def metric_cov(a, r, th):
    """g_{mu nu} in Boyer-Lindquist (t, r, theta, phi), eq. (1), M = 1."""
    Sigma = r * r + a * a * np.cos(th) ** 2
    Delta = r * r - 2.0 * r + a * a
    s2 = np.sin(th) ** 2
    g = np.zeros((4, 4))
    g[0, 0] = -(1.0 - 2.0 * r / Sigma)
    g[0, 3] = g[3, 0] = -2.0 * a * r * s2 / Sigma          # half of the dt dphi coefficient
    g[1, 1] = Sigma / Delta
    g[2, 2] = Sigma
    g[3, 3] = (r * r + a * a + 2.0 * a * a * r * s2 / Sigma) * s2
    return g


def hamiltonian_numeric(a, x, p):
    """H = 1/2 g^{mu nu} p_mu p_nu with the inverse taken numerically. x = (t, r, th, ph), p covariant."""
    ginv = np.linalg.inv(metric_cov(a, x[1], x[2]))
    return 0.5 * p @ ginv @ p


@functools.lru_cache(maxsize=None)
def _symbolic():
    a, r, th, pt, pr, pth, pph = sp.symbols("a r theta p_t p_r p_theta p_phi", real=True)
    Sigma = r ** 2 + a ** 2 * sp.cos(th) ** 2
    Delta = r ** 2 - 2 * r + a ** 2
    s2 = sp.sin(th) ** 2
    g = sp.zeros(4, 4)
    g[0, 0] = -(1 - 2 * r / Sigma)
    g[0, 3] = g[3, 0] = -2 * a * r * s2 / Sigma
    g[1, 1] = Sigma / Delta
    g[2, 2] = Sigma
    g[3, 3] = (r ** 2 + a ** 2 + 2 * a ** 2 * r * s2 / Sigma) * s2
    ginv = g.inv()
    p = sp.Matrix([pt, pr, pth, pph])
    H = sp.Rational(1, 2) * (p.T * ginv * p)[0, 0]
    args = (a, r, th, pt, pr, pth, pph)
    exprs = [sp.diff(H, pt), sp.diff(H, pr), sp.diff(H, pth), sp.diff(H, pph), -sp.diff(H, r), -sp.diff(H, th), H]
    return sp.lambdify(args, exprs, modules="mpmath"), sp.lambdify(args, exprs, modules="numpy")


def hamilton_rhs(a, r, th, pt, pr, pth, pph, high_precision=False):
    """(tdot, rdot, thdot, phdot, prdot, pthdot, H) from Hamilton's equations of H = 1/2 g^{mu nu}p_mu p_nu,
    derived symbolically from eq. (1)."""
    f_mp, f_np = _symbolic()
    if high_precision:
        import mpmath
        with mpmath.workdps(40):
            vals = f_mp(*[mpmath.mpf(float(v)) for v in (a, r, th, pt, pr, pth, pph)])
            return np.array([float(v) for v in vals])
    return np.array(f_np(a, r, th, pt, pr, pth, pph), dtype=float)


# --- closed forms of Kerr photon orbits (Bardeen 1973; Chandrasekhar 1983, cited PAPER.md:L94, L219) ---
def horizon(a):
    return 1.0 + np.sqrt(1.0 - a * a)


def photon_orbit_radii(a):
    """Equatorial circular photon orbits: prograde, retrograde."""
    return (2.0 * (1.0 + np.cos(2.0 / 3.0 * np.arccos(-a))),
            2.0 * (1.0 + np.cos(2.0 / 3.0 * np.arccos(a))))


def critical_xi_eta(a, r):
    """Impact parameters xi = L_z/E, eta = Q/E^2 of the spherical photon orbit of radius r."""
    xi = -(r ** 3 - 3.0 * r ** 2 + a * a * r + a * a) / (a * (r - 1.0))
    eta = -(r ** 3) * (r ** 3 - 6.0 * r ** 2 + 9.0 * r - 4.0 * a * a) / (a * a * (r - 1.0) ** 2)
    return xi, eta


def radial_potential_roots(a, lam, q):
    """Real roots of R(r) = (r^2 + a^2 - a lam)^2 - Delta [(lam - a)^2 + q]  (E = 1)."""
    coeffs = [1.0, 0.0, a * a - lam * lam - q, 2.0 * ((lam - a) ** 2 + q), -a * a * q]
    roots = np.roots(coeffs)
    return np.sort(roots[np.abs(roots.imag) < 1e-9 * (1.0 + np.abs(roots.real))].real)


def captured_closed_form(a, lam, q):
    """A photon arriving from far away is captured iff R(r) has no real root outside the horizon."""
    roots = radial_potential_roots(a, lam, q)
    return not np.any(roots > horizon(a))
