"""Independent end-to-end reference for a RIAF pixel (test helper; not part of the oracle, not part of the product).

Computes the observed intensity I_nu of one image-plane point WITHOUT anything of the oracle: no oracle stepper,
no event logic, no coefficient caching, no oracle formula.

  camera     positions and ray velocities of PAPER.md eqs. (18)-(26); the covariant momentum is then p_mu =
             g_{mu nu} xdot^nu with tdot from the null condition of the metric (1) — not eqs. (7), (8), (4), (5).
  geodesic   scipy DOP853 on Hamilton's equations of H = 1/2 g^{mu nu} p_mu p_nu derived symbolically from
             eq. (1) (tests/kerr_reference.py), all eight components, to the capture / escape surface.
  transfer   eqs. (30), (31) as two more components of that system: dtau/dlambda = r_g alpha_0 / gamma,
             dI/dlambda = r_g j_0 / (gamma nu_0^3) exp(-tau)  (readings C, D), nu_0 = nu / gamma.
  gamma      eq. (2) with a four-velocity built from the metric: Keplerian shells outside the ISCO (reading N),
             inside it the equatorial geodesic with the ISCO's u_t, u_phi obtained by raising indices with the
             numerically inverted metric.
  j, alpha   eqs. (37)-(39) with scipy's K_2, Kirchhoff's law with the Planck function, the plasma of
             BASELINE.json:configs[2]; physical constants typed here from CODATA 2018.
"""
import math

import numpy as np
from scipy import special
from scipy.integrate import solve_ivp

import kerr_reference as K

C, GMSUN, H, KB = 2.99792458e10, 1.3271244e26, 6.62607015e-27, 1.380649e-16
ME, MP, QE = 9.1093837015e-28, 1.67262192369e-24, 4.80320471257e-10


def isco(a):
    """Bardeen, Press & Teukolsky (1972), prograde."""
    z1 = 1 + (1 - a * a) ** (1 / 3) * ((1 + a) ** (1 / 3) + (1 - a) ** (1 / 3))
    z2 = math.sqrt(3 * a * a + z1 * z1)
    return 3 + z2 - math.copysign(1.0, a) * math.sqrt((3 - z1) * (3 + z1 + 2 * z2))


def camera(sc, x, y):
    """Image-plane point -> (r, th, ph) and covariant momentum normalised to p_t = +1 (the ray is traced backwards:
    k = -p_phys, E = -1; readings B, C)."""
    a, ro, to, po = sc["a"], sc["r_obs"], sc["theta_obs"], sc["phi_obs"]
    D = math.sqrt(ro * ro + a * a) * math.sin(to) - y * math.cos(to)          # eqs. (18), (19), z = 0
    xp = D * math.cos(po) - x * math.sin(po)
    yp = D * math.sin(po) + x * math.cos(po)
    zp = ro * math.cos(to) + y * math.sin(to)
    w = xp * xp + yp * yp + zp * zp - a * a
    r = math.sqrt(0.5 * (w + math.sqrt(w * w + 4 * a * a * zp * zp)))          # eq. (20)
    th, ph = math.acos(zp / r), math.atan2(yp, xp)                             # eqs. (21), (22)
    R, Sig, Phi = math.sqrt(r * r + a * a), r * r + a * a * math.cos(th) ** 2, ph - po
    rd = -(r * R * math.sin(th) * math.sin(to) * math.cos(Phi) + R * R * math.cos(th) * math.cos(to)) / Sig   # (24)
    td = (r * math.sin(th) * math.cos(to) - R * math.cos(th) * math.sin(to) * math.cos(Phi)) / Sig           # (25)
    pd = math.sin(to) * math.sin(Phi) / (R * math.sin(th))                                                    # (26)
    g = K.metric_cov(a, r, th)
    # null condition g_tt T^2 + 2 g_tphi T pd + (g_rr rd^2 + g_thth td^2 + g_phph pd^2) = 0 for T = tdot
    A, B2, Cc = g[0, 0], g[0, 3] * pd, g[1, 1] * rd * rd + g[2, 2] * td * td + g[3, 3] * pd * pd
    roots = [(-B2 + s * math.sqrt(B2 * B2 - A * Cc)) / A for s in (1.0, -1.0)]
    for T in roots:
        p = g @ np.array([T, rd, td, pd])
        if p[0] > 0:                                                           # p_t = -E = +1 after normalisation
            return (r, th, ph), p / p[0]
    raise AssertionError("no root with p_t > 0")


class Flow:
    def __init__(self, a):
        self.a, self.r_isco = a, isco(a)
        r = self.r_isco
        den = r ** 0.75 * math.sqrt(r ** 1.5 - 3 * math.sqrt(r) + 2 * a)
        self.E, self.L = (r ** 1.5 - 2 * math.sqrt(r) + a) / den, (r * r - 2 * a * math.sqrt(r) + a * a) / den

    def velocity(self, r, th):
        """u^mu (t, r, th, ph) of reading N, normalised with eq. (1)'s metric at (r, th)."""
        a, g = self.a, K.metric_cov(self.a, r, th)
        ur = 0.0
        if r >= self.r_isco:
            Om = 1.0 / (r ** 1.5 + a)
        else:
            ge = K.metric_cov(a, r, math.pi / 2)
            up = np.linalg.inv(ge) @ np.array([-self.E, 0.0, 0.0, self.L])      # equatorial geodesic, indices raised
            Om = up[3] / up[0]
            ur2 = (-1.0 - (ge[0, 0] * up[0] ** 2 + 2 * ge[0, 3] * up[0] * up[3] + ge[3, 3] * up[3] ** 2)) / ge[1, 1]
            ur = -math.sqrt(max(ur2, 0.0))
        # u = u^t (1, 0, 0, Om) + (0, u^r, 0, 0),  g(u, u) = -1
        N = -(g[0, 0] + 2 * Om * g[0, 3] + Om * Om * g[3, 3])
        if N <= 0:
            return None
        ut = math.sqrt((1.0 + g[1, 1] * ur * ur) / N)
        return np.array([ut, ur, 0.0, ut * Om])


def coefficients(md, a, r, th, nu0):
    """j_nu0 (per steradian: reading F) and alpha_nu0 in cgs, eqs. (37)-(39) + Kirchhoff."""
    rh = K.horizon(a)
    ne = md["n0"] * (r / rh) ** md["n_index"] * math.exp(-math.cos(th) ** 2 / (2 * md["h_over_r"] ** 2))
    Te = md["T0"] * (r / rh) ** md["T_index"]
    Bf = math.sqrt(8 * math.pi * ne * MP * C * C / (6 * md["beta"] * r))
    Th = KB * Te / (ME * C * C)
    nuc = 3 * QE * Bf / (4 * math.pi * ME * C) * Th * Th
    xM = nu0 / nuc
    Mx = 4.0505 / xM ** (1 / 6) * (1 + 0.40 / xM ** 0.25 + 0.5316 / xM ** 0.5) * math.exp(-1.8899 * xM ** (1 / 3))
    K2 = special.kv(2, 1.0 / Th)
    if not (Mx > 0 and K2 > 0):
        return 0.0, 0.0
    j = md["j_scale"] * nu0 * ne * QE * QE * Mx / (math.sqrt(3) * C * K2)
    xp = H * nu0 / (KB * Te)
    Bnu = 2 * H * nu0 ** 3 / (C * C) / math.expm1(xp) if xp < 700 else 0.0
    return j, (j / Bnu if Bnu > 0 else 0.0)


def pixel(sc, md, nus, x, y, rtol=1e-10):
    """I_nu [len(nus)], tau [len(nus)], flag ('captured' / 'escaped'), end state of the ray through (x, y)."""
    a, nf = sc["a"], len(nus)
    (r0, th0, ph0), p0 = camera(sc, x, y)
    flow = Flow(a)
    rg = GMSUN * md["mbh_msun"] / (C * C)
    r_cap = K.horizon(a) + sc["horizon_eps"]

    def f(lam, s):
        t, r, th, ph, pt, pr, pth, pph = s[:8]
        d = K.hamilton_rhs(a, r, th, pt, pr, pth, pph)
        out = [d[0], d[1], d[2], d[3], 0.0, d[4], d[5], 0.0] + [0.0] * (2 * nf)
        if r_cap < r < md["r_rt_out"]:
            u = flow.velocity(r, th)
            if u is not None:
                ig = u[0] * pt + u[1] * pr + u[3] * pph                        # 1/gamma = k_alpha u^alpha (eq. (2), E = -1)
                if ig > 0 and math.isfinite(ig):
                    gam = 1.0 / ig
                    for k, nu in enumerate(nus):
                        j, al = coefficients(md, a, r, th, nu / gam)
                        out[8 + k] = rg * al / gam
                        out[8 + nf + k] = rg * j / (gam * (nu / gam) ** 3) * math.exp(-s[8 + k])
        return out

    def captured(lam, s):
        return s[1] - r_cap
    captured.terminal, captured.direction = True, -1.0

    def escaped(lam, s):
        return s[1] - sc["r_esc"] if s[5] > 0 else -1.0
    escaped.terminal, escaped.direction = True, 1.0
    s0 = [0.0, r0, th0, ph0, p0[0], p0[1], p0[2], p0[3]] + [0.0] * (2 * nf)
    atol = [1e-12] * 8 + [1e-14] * nf + [1e-80] * nf            # (the invariant intensity is ~1e-40 in cgs)
    sol = solve_ivp(f, [0.0, 6000.0], s0, method="DOP853", rtol=rtol, atol=atol, events=[captured, escaped], max_step=50.0)
    assert sol.status == 1, "ray reached neither surface"
    end = sol.y[:, -1]
    nus = np.asarray(nus, float)
    return nus ** 3 * end[8 + nf:8 + 2 * nf], end[8:8 + nf], ("captured" if len(sol.t_events[0]) else "escaped"), end[:8]
