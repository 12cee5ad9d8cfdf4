// odyssey_oracle.cpp — plain, slow, FP64 CPU ORACLE for the Odyssey hot path (arXiv 1601.02063).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header, table
// or constant generator with the CUDA path in paper_1601_02063_b200/csrc/, and neither side
// includes or imports the other.
//
// What it computes: one ray per image-plane pixel, traced backwards from the observer through the
// Kerr spacetime in Boyer–Lindquist coordinates (§2.1, eqs. (1)-(15)), initial conditions
// of PAPER.md §2.2 (eqs. (18)-(26), (7), (8), (4), (5), (13)), adaptive embedded 5th-order
// Runge–Kutta with step control "after Press et al. 1992", with the radiative
// transfer of PAPER.md §2.3 (eqs. (2), (27)-(31)) advanced once per accepted step, and the
// emission models of PAPER.md §4.3 (thin Keplerian disk) and §4.5 (thermal synchrotron,
// eqs. (37)-(39)) with the flow profile of BASELINE.json:configs[2].
//
// It follows the algorithm step by step, one ray at a time, in the paper's notation; there is no
// blocking, fusion, vectorisation or reordering.  The only parallelism is an OpenMP loop over
// independent pixels in the image drivers at the bottom.  Readings taken where the paper is
// silent, ambiguous or garbled are labelled [reading X] and listed in DESIGN.md §3 (they are
// SURVEY.md §8(c)'s rows A..T).
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): RHS vs finite-difference Hamilton equations of
// a numerically inverted metric (1); printed eqs. (14),(15) on shell; H = 0, eqs. (16),(17) and the
// a = 0 closed forms at the start; tableau order conditions and observed order 5; drift of Q and of
// the null condition; capture classification vs the closed-form radial potential; shadow edges
// sqrt(27) and Bardeen's xi(r_ph); Schwarzschild deflection vs quadrature; an independent
// 8-component scipy integration of Hamilton's equations (E, L_z drift there); closed-form Keplerian
// g; uniform-slab RT; the thin limit and the formal solution int eps e^-tau dlambda by independent
// quadrature on a finer path; K_2 vs scipy; M(1) as printed in eq. (38).
// The RIAF images and the SED as a whole (oracle_render_image kind 2, oracle_render_spectrum) have no value
// printed in the paper to compare with (Figs. 9, 10 are pictures, Broderick & Loeb's table is not in the
// container); they are pinned end to end by tests/test_oracle_riaf_independent.py against a computation that
// shares nothing with this file (tests/riaf_reference.py: momenta from the metric and the null condition, scipy
// DOP853 on the symbolically derived 8-component Hamiltonian system with eqs. (30), (31) as two more components,
// scipy's K_2): pixels of C2 thin and thick, captured, escaping and frozen, to the truncation level of reading E
// (3e-3 at rtol 1e-8, converging: 6e-5 at 1e-12), a five-frequency SED, and a scene whose first and event-
// located last step carry weight.
//
// Build: g++ -std=c++17 -O2 -fopenmp -fPIC -shared (see oracle/build.py).  -ffast-math is never used.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ----------------------------------------------------------------------------------------------
// Physical constants, cgs (CODATA 2018; G M_sun from the IAU nominal solar mass parameter).
// ----------------------------------------------------------------------------------------------
constexpr double C_LIGHT = 2.99792458e10;        // cm/s
constexpr double GM_SUN  = 1.3271244e26;         // cm^3/s^2
constexpr double H_PLANCK = 6.62607015e-27;      // erg s
constexpr double K_BOLTZ = 1.380649e-16;         // erg/K
constexpr double M_ELECTRON = 9.1093837015e-28;  // g
constexpr double M_PROTON = 1.67262192369e-24;   // g
constexpr double E_CHARGE = 4.80320471257e-10;   // esu
constexpr double PI = 3.14159265358979323846;
constexpr double G_NEWTON = 6.67430e-8;          // cm^3 g^-1 s^-2
constexpr double SIGMA_SB = 5.670374419e-5;      // erg cm^-2 s^-1 K^-4

enum Flag { ESCAPED = 0, CAPTURED = 1, DISK = 2, OPAQUE = 3, MAXSTEP = 4 };

struct Scene {           // mirrors workloads.scene(); plain C layout, see oracle/binding.py
    double a, r_obs, theta_obs, phi_obs;
    double x_min, x_max, y_min, y_max;
    int32_t nx, ny;
    double rtol;
    int32_t tableau, pad0;
    double h0, horizon_eps, r_esc;
    int32_t max_attempts, pad1;
};

struct Model {           // mirrors workloads.model_*()
    int32_t kind, nbins;
    double r_in, r_out, emis_index;
    double mbh_msun, n0, n_index, T0, T_index, h_over_r, beta, r_rt_out, tau_max, j_scale;
    double g_lo, g_hi, g_power;
    int32_t rt_scheme, pad;  // 0: one update per accepted step [reading E]; 1: tau, I as Runge-Kutta components [E']
    double spot_r_orbit, spot_size, spot_phi0;   // kind 3 [reading HS]: orbit radius (<= 0: r_isco), r_spot, azimuth at t = 0
    double mdot_gs;                              // kind 4 [reading NT]: accretion rate, g/s
    double dtau_max;                             // kind 2, rt_scheme 0 [reading DT]: cap of the next step's optical depth (<= 0: off)
};

// ----------------------------------------------------------------------------------------------
// Kerr helpers (M = 1).
// ----------------------------------------------------------------------------------------------
double horizon_radius(double a) { return 1.0 + std::sqrt(1.0 - a * a); }

// Marginally stable orbit of Bardeen, Press & Teukolsky 1972 (cited PAPER.md:L223) for an orbit in
// the +phi direction around a hole of signed spin a.
double isco_radius(double a) {
    double z1 = 1.0 + std::cbrt(1.0 - a * a) * (std::cbrt(1.0 + a) + std::cbrt(1.0 - a));
    double z2 = std::sqrt(3.0 * a * a + z1 * z1);
    double s = (a >= 0.0) ? 1.0 : -1.0;
    return 3.0 + z2 - s * std::sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2));
}

// Energy and angular momentum per unit mass of the circular equatorial orbit at radius r (+phi).
void circular_orbit_EL(double a, double r, double* E, double* L) {
    double sr = std::sqrt(r);
    double den = std::pow(r, 0.75) * std::sqrt(r * sr - 3.0 * sr + 2.0 * a);
    *E = (r * sr - 2.0 * sr + a) / den;
    *L = (r * r - 2.0 * a * sr + a * a) / den;
}

// ----------------------------------------------------------------------------------------------
// Ray = constants of motion of one geodesic.  E = -1 always after normalisation [reading B, C].
// State y = (r, theta, phi, p_r, p_theta)  (t is not needed by any output; PAPER.md:L88 lists it).
// ----------------------------------------------------------------------------------------------
struct Ray { double a, E, L, Q; };
constexpr int NV = 6;      // y = (r, theta, phi, p_r, p_theta, t): the six parameters of PAPER.md:L88; t does not enter the error norm

// Steps 1-4: pixel -> Boyer-Lindquist position, velocity, constants, momenta.  PAPER.md:L104-143.
// raw[0..1] receive E^2 and L_z BEFORE the |E| normalisation (for the closed-form pins).
void init_ray(const Scene& S, double x, double y, Ray* ray, double st[NV], double raw[2]) {
    const double a = S.a, z = 0.0;
    const double so = std::sin(S.theta_obs), co = std::cos(S.theta_obs);
    const double sp = std::sin(S.phi_obs), cp = std::cos(S.phi_obs);
    // eq. (19), (18)
    double D = (std::sqrt(S.r_obs * S.r_obs + a * a) - z) * so - y * co;
    double xp = D * cp - x * sp;
    double yp = D * sp + x * cp;
    double zp = (S.r_obs - z) * co + y * so;
    // eqs. (20)-(22)
    double w = xp * xp + yp * yp + zp * zp - a * a;
    double r = std::sqrt((w + std::sqrt(w * w + 4.0 * a * a * zp * zp)) / 2.0);
    double th = std::acos(zp / r);
    double ph = std::atan2(yp, xp);
    // eqs. (24)-(26)
    double R = std::sqrt(r * r + a * a);
    double Phi = ph - S.phi_obs;
    double s = std::sin(th), c = std::cos(th);
    double Sigma = r * r + a * a * c * c;
    double Delta = r * r - 2.0 * r + a * a;
    double rdot = -(r * R * s * so * std::cos(Phi) + R * R * c * co) / Sigma;
    double thdot = (r * s * co - R * c * so * std::cos(Phi)) / Sigma;
    double phdot = so * std::sin(Phi) / (R * s);
    // eq. (7) with mu = 0; E = -sqrt(E^2): the ray is traced backwards in time [reading B]
    double E2 = ((Sigma - 2.0 * r) / (Sigma * Delta)) * (Sigma * rdot * rdot + Sigma * Delta * thdot * thdot)
              + Delta * phdot * phdot * s * s;
    double E = -std::sqrt(E2);
    // eq. (8)
    double L = (Sigma * Delta * phdot - 2.0 * a * r * E) * s * s / (Sigma - 2.0 * r);
    // eqs. (4), (5)
    double pr = Sigma * rdot / Delta;
    double pth = Sigma * thdot;
    if (raw) { raw[0] = E2; raw[1] = L; }
    // normalise so that |E| = 1: the affine parameter is then length in r_g far away [reading C]
    double n = std::fabs(E);
    L /= n; pr /= n; pth /= n; E = -1.0;
    // eq. (13) with mu = 0
    double Q = pth * pth + (L * L / (s * s) - a * a * E * E) * c * c;
    ray->a = a; ray->E = E; ray->L = L; ray->Q = Q;
    st[0] = r; st[1] = th; st[2] = ph; st[3] = pr; st[4] = pth; st[5] = 0.0;   // coordinate time counted from the observer
}

// Step 5: right-hand side.  rdot, thetadot from (4),(5); phidot (12); pdot_r, pdot_theta are
// -dH/dr, -dH/dtheta of H = G/(2 Sigma) WITHOUT the null constraint substituted [reading A]; on
// G = 0 they are eqs. (14),(15).  Pole clamp of PAPER.md:L90 [reading I].
void rhs(const Ray& ray, const double y[NV], double dy[NV]) {
    const double a = ray.a, E = ray.E, L = ray.L;
    const double r = y[0], th = y[1], pr = y[3], pth = y[4];
    double s = std::sin(th), c = std::cos(th);
    if (std::fabs(s) < 1e-8) s = std::copysign(1e-8, s);
    double Sigma = r * r + a * a * c * c;
    double Delta = r * r - 2.0 * r + a * a;
    double P = (r * r + a * a) * E - a * L;
    double D = L / s - a * E * s;
    double G = Delta * pr * pr + pth * pth + D * D - P * P / Delta;   // = 2 Sigma H
    dy[0] = Delta * pr / Sigma;
    dy[1] = pth / Sigma;
    dy[2] = (2.0 * a * r * E + (Sigma - 2.0 * r) * L / (s * s)) / (Sigma * Delta);
    dy[3] = -((r - 1.0) * pr * pr - 2.0 * r * E * P / Delta + (r - 1.0) * P * P / (Delta * Delta)) / Sigma
            + r * G / (Sigma * Sigma);
    dy[4] = s * c * (L * L / (s * s * s * s) - a * a * E * E) / Sigma - a * a * s * c * G / (Sigma * Sigma);
    dy[5] = E + (2.0 * r * (r * r + a * a) * E - 2.0 * a * r * L) / (Sigma * Delta);                      // eq. (9)
}

// Scale-free null-condition residual [reading R]: G over the sum of the magnitudes of its terms.
double null_ratio(const Ray& ray, const double y[5]) {
    const double a = ray.a, E = ray.E, L = ray.L;
    double s = std::sin(y[1]);
    if (std::fabs(s) < 1e-8) s = std::copysign(1e-8, s);
    double Delta = y[0] * y[0] - 2.0 * y[0] + a * a;
    double P = (y[0] * y[0] + a * a) * E - a * L;
    double D = L / s - a * E * s;
    double t1 = Delta * y[3] * y[3], t2 = y[4] * y[4], t3 = D * D, t4 = P * P / Delta;
    return (t1 + t2 + t3 - t4) / (std::fabs(t1) + t2 + t3 + std::fabs(t4));
}

// Carter constant from the current state, eq. (13) with mu = 0.
double carter_Q(const Ray& ray, const double y[5]) {
    double s = std::sin(y[1]), c = std::cos(y[1]);
    return y[4] * y[4] + (ray.L * ray.L / (s * s) - ray.a * ray.a * ray.E * ray.E) * c * c;
}

// ----------------------------------------------------------------------------------------------
// Step 6: embedded 6-stage Runge-Kutta 5(4) pairs [reading H].
// ----------------------------------------------------------------------------------------------
struct Tableau { double c[6], A[6][6], b5[6], b4[6]; };

Tableau make_tableau(int which) {
    Tableau T;
    std::memset(&T, 0, sizeof(T));
    if (which == 0) {          // Fehlberg 4(5), BASELINE.json:configs[0] "RKF45"
        const double c[6] = {0.0, 1.0 / 4, 3.0 / 8, 12.0 / 13, 1.0, 1.0 / 2};
        std::memcpy(T.c, c, sizeof(c));
        T.A[1][0] = 1.0 / 4;
        T.A[2][0] = 3.0 / 32;        T.A[2][1] = 9.0 / 32;
        T.A[3][0] = 1932.0 / 2197;   T.A[3][1] = -7200.0 / 2197;  T.A[3][2] = 7296.0 / 2197;
        T.A[4][0] = 439.0 / 216;     T.A[4][1] = -8.0;            T.A[4][2] = 3680.0 / 513;    T.A[4][3] = -845.0 / 4104;
        T.A[5][0] = -8.0 / 27;       T.A[5][1] = 2.0;             T.A[5][2] = -3544.0 / 2565;  T.A[5][3] = 1859.0 / 4104;  T.A[5][4] = -11.0 / 40;
        const double b5[6] = {16.0 / 135, 0.0, 6656.0 / 12825, 28561.0 / 56430, -9.0 / 50, 2.0 / 55};
        const double b4[6] = {25.0 / 216, 0.0, 1408.0 / 2565, 2197.0 / 4104, -1.0 / 5, 0.0};
        std::memcpy(T.b5, b5, sizeof(b5));
        std::memcpy(T.b4, b4, sizeof(b4));
    } else {                   // Cash-Karp, the pair used by Press et al. 1992
        const double c[6] = {0.0, 1.0 / 5, 3.0 / 10, 3.0 / 5, 1.0, 7.0 / 8};
        std::memcpy(T.c, c, sizeof(c));
        T.A[1][0] = 1.0 / 5;
        T.A[2][0] = 3.0 / 40;          T.A[2][1] = 9.0 / 40;
        T.A[3][0] = 3.0 / 10;          T.A[3][1] = -9.0 / 10;      T.A[3][2] = 6.0 / 5;
        T.A[4][0] = -11.0 / 54;        T.A[4][1] = 5.0 / 2;        T.A[4][2] = -70.0 / 27;       T.A[4][3] = 35.0 / 27;
        T.A[5][0] = 1631.0 / 55296;    T.A[5][1] = 175.0 / 512;    T.A[5][2] = 575.0 / 13824;    T.A[5][3] = 44275.0 / 110592;  T.A[5][4] = 253.0 / 4096;
        const double b5[6] = {37.0 / 378, 0.0, 250.0 / 621, 125.0 / 594, 0.0, 512.0 / 1771};
        const double b4[6] = {2825.0 / 27648, 0.0, 18575.0 / 48384, 13525.0 / 55296, 277.0 / 14336, 1.0 / 4};
        std::memcpy(T.b5, b5, sizeof(b5));
        std::memcpy(T.b4, b4, sizeof(b4));
    }
    return T;
}

// One attempt of size h from y: 5th-order result ynew and the error estimate yerr = 5th - 4th,
// formed as h * sum (b5_j - b4_j) k_j exactly as Press et al.'s rkck does.
// ystage (optional) receives the six stage states y + h sum_j A_ij k_j.
void rk_attempt(const Ray& ray, const Tableau& T, const double y[NV], double h, double ynew[NV], double yerr[NV],
                double (*ystage)[NV] = nullptr) {
    double k[6][NV], ytmp[NV];
    for (int i = 0; i < 6; ++i) {
        for (int v = 0; v < NV; ++v) {
            double acc = 0.0;
            for (int j = 0; j < i; ++j) acc += T.A[i][j] * k[j][v];
            ytmp[v] = y[v] + h * acc;
            if (ystage) ystage[i][v] = ytmp[v];
        }
        rhs(ray, ytmp, k[i]);
    }
    for (int v = 0; v < NV; ++v) {
        double s5 = 0.0, se = 0.0;
        for (int j = 0; j < 6; ++j) { s5 += T.b5[j] * k[j][v]; se += (T.b5[j] - T.b4[j]) * k[j][v]; }
        ynew[v] = y[v] + h * s5;
        yerr[v] = h * se;
    }
}

// Step 7: scaled max-norm of the error in units of rtol [reading G].
double error_norm(const double y[NV], const double yerr[NV], double rtol) {     // over (r, theta, phi, p_r, p_theta) only
    const double sc[5] = {std::fabs(y[0]), 1.0, 1.0, 1.0 + std::fabs(y[3]), 1.0 + std::fabs(y[4])};
    double e = 0.0;
    for (int v = 0; v < 5; ++v) {
        double q = std::fabs(yerr[v]) / sc[v];
        if (q > e || std::isnan(q)) e = q;    // a NaN sticks: every later comparison with it is false
    }
    return e / rtol;
}

// ----------------------------------------------------------------------------------------------
// Step 10: flow four-velocity and energy-shift factor gamma of eq. (2) [reading N].
// ----------------------------------------------------------------------------------------------
struct Flow { double r_isco, E_isco, L_isco; };

Flow make_flow(double a) {
    Flow F;
    F.r_isco = isco_radius(a);
    circular_orbit_EL(a, F.r_isco, &F.E_isco, &F.L_isco);
    return F;
}

// u = (ut, ur, 0, uphi) at (r, theta).  Returns false where the normalisation has no solution.
bool flow_velocity(double a, const Flow& F, double r, double th, double u[4]) {
    double s = std::sin(th), c = std::cos(th);
    double s2 = s * s;
    double Sigma = r * r + a * a * c * c;
    double Delta = r * r - 2.0 * r + a * a;
    // covariant metric, eq. (1)
    double g_tt = -(1.0 - 2.0 * r / Sigma);
    double g_tp = -2.0 * a * r * s2 / Sigma;
    double g_pp = (r * r + a * a + 2.0 * a * a * r * s2 / Sigma) * s2;
    double g_rr = Sigma / Delta;
    double Omega, ur;
    if (r >= F.r_isco) {                    // Keplerian shells, u^theta = 0
        Omega = 1.0 / (r * std::sqrt(r) + a);
        ur = 0.0;
    } else {                                // plunging: the equatorial geodesic with (E, L) of the ISCO
        double E = F.E_isco, L = F.L_isco;
        double ut_eq = ((r * r + a * a + 2.0 * a * a / r) * E - (2.0 * a / r) * L) / Delta;
        double up_eq = ((2.0 * a / r) * E + (1.0 - 2.0 / r) * L) / Delta;
        Omega = up_eq / ut_eq;
        double ur2 = E * E - 1.0 + 2.0 / r - (L * L - a * a * (E * E - 1.0)) / (r * r)
                   + 2.0 * (L - a * E) * (L - a * E) / (r * r * r);
        if (ur2 < 0.0) ur2 = 0.0;
        ur = -std::sqrt(ur2);
    }
    double N = -(g_tt + 2.0 * Omega * g_tp + Omega * Omega * g_pp);
    if (!(N > 0.0)) return false;
    double ut = std::sqrt((1.0 + g_rr * ur * ur) / N);
    u[0] = ut; u[1] = ur; u[2] = 0.0; u[3] = Omega * ut;
    return true;
}

// eq. (2): gamma = (k_alpha u^alpha)_inf / (k_alpha u^alpha)_lambda with k_t = -E = 1 at infinity
// for a static observer, k_r = p_r, k_theta = p_theta, k_phi = L.
double gamma_shift(const Ray& ray, const double y[5], const double u[4]) {
    double k_t = -ray.E;
    return k_t / (k_t * u[0] + y[3] * u[1] + y[4] * u[2] + ray.L * u[3]);
}

// ----------------------------------------------------------------------------------------------
// Step 11: plasma state and thermal synchrotron coefficients, eqs. (37)-(39) [readings F, O].
// ----------------------------------------------------------------------------------------------
double bessel_K2(double x) { return std::cyl_bessel_k(2.0, x); }

double mahadevan_M(double xM) {           // eq. (38)
    return 4.0505 / std::pow(xM, 1.0 / 6.0)
         * (1.0 + 0.40 / std::pow(xM, 0.25) + 0.5316 / std::sqrt(xM))
         * std::exp(-1.8899 * std::cbrt(xM));
}

double planck_B(double nu, double T) {    // B_nu(T), cgs
    return (2.0 * H_PLANCK * nu * nu * nu / (C_LIGHT * C_LIGHT)) / std::expm1(H_PLANCK * nu / (K_BOLTZ * T));
}

struct Plasma { double n_e, T_e, B, Theta_e, nu_c; };

Plasma plasma_state(const Model& M, double a, double r, double th) {
    Plasma p;
    double rh = horizon_radius(a);
    double c = std::cos(th);
    p.n_e = M.n0 * std::pow(r / rh, M.n_index) * std::exp(-c * c / (2.0 * M.h_over_r * M.h_over_r));
    p.T_e = M.T0 * std::pow(r / rh, M.T_index);
    p.B = std::sqrt(8.0 * PI * p.n_e * M_PROTON * C_LIGHT * C_LIGHT / (6.0 * M.beta * r));
    p.Theta_e = K_BOLTZ * p.T_e / (M_ELECTRON * C_LIGHT * C_LIGHT);
    p.nu_c = (3.0 * E_CHARGE * p.B / (4.0 * PI * M_ELECTRON * C_LIGHT)) * p.Theta_e * p.Theta_e;   // eq. (39)
    return p;
}

// j_nu0 per steradian (eq. (37) without its 4 pi; j_scale = 4 pi restores the print) and alpha by
// Kirchhoff's law, both at the local frequency nu0.
void synchrotron_coefficients(const Model& M, const Plasma& p, double nu0, double* j, double* alpha) {
    double xM = nu0 / p.nu_c;
    double Mx = mahadevan_M(xM);
    double K2 = bessel_K2(1.0 / p.Theta_e);
    double jj = 0.0;
    if (Mx > 0.0 && K2 > 0.0)
        jj = M.j_scale * nu0 * p.n_e * E_CHARGE * E_CHARGE * Mx / (std::sqrt(3.0) * C_LIGHT * K2);
    double Bnu = planck_B(nu0, p.T_e);
    *j = jj;
    *alpha = (jj > 0.0 && Bnu > 0.0) ? jj / Bnu : 0.0;
}

// Coefficients of eqs. (30),(31) per unit affine parameter at one point of the ray, for each
// frequency k [readings C, D]:  a_k = r_g alpha_0(nu_0)/gamma,  eps_k = r_g j_0(nu_0)/(gamma nu_0^3),
// nu_0 = nu_k/gamma.  Zero outside horizon+eps < r < r_rt_out or where the flow
// has no velocity.
void rt_coefficients(const Scene& S, const Model& M, const Flow& F, const Ray& ray, const double y[5],
                     int nf, const double* nu, double* acoef, double* ecoef) {
    for (int k = 0; k < nf; ++k) { acoef[k] = 0.0; ecoef[k] = 0.0; }
    double r = y[0];
    if (!(r > horizon_radius(S.a) + S.horizon_eps && r < M.r_rt_out)) return;
    double u[4];
    if (!flow_velocity(S.a, F, r, y[1], u)) return;
    double gam = gamma_shift(ray, y, u);
    if (!(gam > 0.0) || !std::isfinite(gam)) return;
    Plasma p = plasma_state(M, S.a, r, y[1]);
    double rg_cm = GM_SUN * M.mbh_msun / (C_LIGHT * C_LIGHT);
    for (int k = 0; k < nf; ++k) {
        double nu0 = nu[k] / gam, j, al;
        synchrotron_coefficients(M, p, nu0, &j, &al);
        acoef[k] = rg_cm * al / gam;
        ecoef[k] = rg_cm * j / (gam * nu0 * nu0 * nu0);
    }
}

// Step 9: one RT update over an accepted step of affine length dl [reading E]: trapezoid in lambda
// for dtau and for the emission, with the exact attenuation across the step,
// phi(x) = (1 - e^-x)/x.  T = exp(-tau) is carried as a product.  A frequency is frozen once
// tau > tau_max.
void rt_update(double a0, double a1, double e0, double e1, double dl, double tau_max,
               double* tau, double* T, double* I) {
    if (*tau > tau_max) return;
    double dtau = 0.5 * (a0 + a1) * dl;
    double phi = (dtau > 0.0) ? -std::expm1(-dtau) / dtau : 1.0;
    *I += *T * 0.5 * (e0 + e1) * dl * phi;
    *T *= std::exp(-dtau);
    *tau += dtau;
}

// Alternative reading [E'] of PAPER.md:L171 ("easily integrated along with the geodesic"): tau and the
// invariant intensity are two more components of the Runge-Kutta system,
//   dtau/dlambda = a(lambda),   dI/dlambda = eps(lambda) exp(-tau(lambda))      (eqs. (30), (31)),
// advanced through the same six stages with the fifth-order weights; they do not enter the error norm
// (the geodesic alone controls the step, so both schemes take identical steps).  a[i], eps[i] are the
// coefficients at the six stage states.  A frequency is frozen once tau > tau_max, as in rt_update.
void rt_rk_step(const Tableau& T, const double a[6], const double eps[6], double h, double tau_max,
                double* tau, double* I) {
    if (*tau > tau_max) return;
    double s_tau = 0.0, s_I = 0.0;
    for (int i = 0; i < 6; ++i) {
        double acc = 0.0;
        for (int j = 0; j < i; ++j) acc += T.A[i][j] * a[j];
        double tau_i = *tau + h * acc;                     // stage value of tau
        s_tau += T.b5[i] * a[i];
        s_I += T.b5[i] * eps[i] * std::exp(-tau_i);
    }
    *I += h * s_I;
    *tau += h * s_tau;
}

// ----------------------------------------------------------------------------------------------
// Step 8 + the per-ray driver.
// ----------------------------------------------------------------------------------------------
struct RayOut {
    int flag; double r, th, ph, t; int n_attempt, n_accept;
    double g, r_e;                       // thin disk
    std::vector<double> I, tau;          // invariant intensity I_nu/nu^3 and optical depth per frequency
};

struct Path {
    std::vector<double> nodes;   // per accepted node: (r, theta, phi, p_r, p_theta), the affine parameter, t
    std::vector<double> absorb;  // per accepted node: invariant absorption coefficient of frequency 0 there (kind 2, nf >= 1)
};

constexpr int LOCATE_MAX = 8;

void trace_ray(const Scene& S, const Model& M, int nf, const double* nu, double x, double yimg,
               RayOut* out, Path* path) {
    Ray ray; double y[NV];
    init_ray(S, x, yimg, &ray, y, nullptr);
    const Tableau T = make_tableau(S.tableau);
    const Flow F = make_flow(S.a);
    const double r_cap = horizon_radius(S.a) + S.horizon_eps;
    double r_in = (M.r_in > 0.0) ? M.r_in : F.r_isco;
    if (M.kind == 3 && !(M.r_in > 0.0)) {
        // [reading HS] PAPER.md:L259 lights everything "within d < 4 r_spot" of a centre that orbits AT r_isco, so the
        // opaque plane must reach inwards to the inner edge of the spot (d is measured in the pseudo-Cartesian radius
        // sqrt(r^2 + a^2) of eqs. (33), (34)); with the thin disk's default (r_isco) the inner half would never be lit.
        const double rs = (M.spot_r_orbit > 0.0) ? M.spot_r_orbit : F.r_isco;
        const double Rin = std::sqrt(rs * rs + S.a * S.a) - 4.0 * M.spot_size;
        r_in = (Rin > std::fabs(S.a)) ? std::sqrt(Rin * Rin - S.a * S.a) : 0.0;
    }
    double h = S.h0;
    int n_attempt = 0, n_accept = 0, flag = -1;
    bool on_equator = false;
    std::vector<double> tau(nf, 0.0), Tr(nf, 1.0), I(nf, 0.0), a0(nf, 0.0), e0(nf, 0.0), a1(nf, 0.0), e1(nf, 0.0);
    double g = 0.0, r_e = 0.0, phi_plane = 0.0;
    if (M.kind == 2) rt_coefficients(S, M, F, ray, y, nf, nu, a0.data(), e0.data());
    double lambda = 0.0;
    if (path) { path->nodes.insert(path->nodes.end(), y, y + 5); path->nodes.push_back(lambda); path->nodes.push_back(y[5]); if (nf > 0) path->absorb.push_back(a0[0]); }

    while (flag < 0) {
        if (n_attempt >= S.max_attempts) { flag = MAXSTEP; break; }
        double ynew[NV], yerr[NV], ystage[6][NV];
        rk_attempt(ray, T, y, h, ynew, yerr, ystage);
        ++n_attempt;
        double err = error_norm(y, yerr, S.rtol);
        if (!(err <= 1.0)) {                               // reject (also when err is NaN)
            if (!std::isfinite(err)) h *= 0.1;
            else h *= std::max(0.1, 0.9 * std::pow(err, -0.25));
            continue;
        }
        ++n_accept;
        double h_used = h;
        double h_next = h * std::min(5.0, 0.9 * std::pow(err, -0.2));

        // Event location: re-take this step from its start state y with h adjusted by Newton until
        // the trial end lies on the surface f = 0 (component comp of the state equal to target).
        auto locate = [&](int comp, double target) {
            double ftol = 1e-12 * std::max(1.0, std::fabs(target));
            for (int it = 0; it < LOCATE_MAX; ++it) {
                double f = ynew[comp] - target;
                if (std::fabs(f) <= ftol) break;
                double dy[NV];
                rhs(ray, ynew, dy);
                // safeguard [reading J]: the Newton update must stay inside (0, ~the accepted step] (h_next >= 0.9 h);
                // a flat or non-finite slope, or a non-finite trial state, halves the step length instead
                double hn = h_used - f / dy[comp];
                h_used = (hn > 0.0 && hn <= 1.2 * h_next) ? hn : 0.5 * h_used;
                rk_attempt(ray, T, y, h_used, ynew, yerr, ystage);
                ++n_attempt;
            }
        };

        // (1) thin disk: equatorial crossing inside the step [reading P]
        if ((M.kind == 1 || M.kind == 3 || M.kind == 4) && !on_equator && std::cos(y[1]) * std::cos(ynew[1]) < 0.0) {
            // A ray that has passed through the axis (possible only for L_z = 0, or when the integrator steps over the
            // centrifugal barrier of a tiny L_z) continues with theta outside [0, pi]: the equatorial plane is
            // theta = pi/2 + k pi, and (r, pi/2 + k pi, phi) is the point (r, pi/2, phi + k pi).
            const double k_eq = std::nearbyint((ynew[1] - 0.5 * PI) / PI);
            locate(1, 0.5 * PI + k_eq * PI);
            on_equator = true;
            if (ynew[0] >= r_in && ynew[0] <= M.r_out && ynew[0] > r_cap) {
                flag = DISK;
                r_e = ynew[0];
                phi_plane = k_eq * PI;
                double u[4];
                double yeq[NV] = {ynew[0], 0.5 * PI, ynew[2], ynew[3], ynew[4], ynew[5]};
                if (flow_velocity(S.a, F, r_e, 0.5 * PI, u)) g = gamma_shift(ray, yeq, u);
            }
        } else {
            on_equator = false;
        }
        // (2) capture, (3) escape — tested on the (possibly truncated) end state [reading J]
        if (flag < 0) {
            if (ynew[0] <= r_cap) { locate(0, r_cap); flag = CAPTURED; }
            else if (ynew[3] > 0.0 && ynew[0] >= S.r_esc) { locate(0, S.r_esc); flag = ESCAPED; }
        }
        // RT over the step actually taken
        if (M.kind == 2 && M.rt_scheme == 0) {
            rt_coefficients(S, M, F, ray, ynew, nf, nu, a1.data(), e1.data());
            bool all_opaque = true;
            for (int k = 0; k < nf; ++k) {
                rt_update(a0[k], a1[k], e0[k], e1[k], h_used, M.tau_max, &tau[k], &Tr[k], &I[k]);
                if (!(tau[k] > M.tau_max)) all_opaque = false;
            }
            a0.swap(a1); e0.swap(e1);
            if (flag < 0 && all_opaque) flag = OPAQUE;
            // [reading DT, SURVEY §8(f)-2 "a Δτ-limited step cap"]: the next step may not be longer than dtau_max
            // optical depths at the absorption coefficient of the point just reached (largest over the frequencies
            // still being integrated)
            if (M.dtau_max > 0.0) {
                double amax = 0.0;
                for (int k = 0; k < nf; ++k) if (!(tau[k] > M.tau_max)) amax = std::max(amax, a0[k]);
                if (amax > 0.0) h_next = std::min(h_next, M.dtau_max / amax);
            }
        } else if (M.kind == 2) {                       // [E']: coefficients at the six stage states of the step taken
            std::vector<double> as(6 * (size_t)nf), es(6 * (size_t)nf);
            for (int i = 0; i < 6; ++i)
                rt_coefficients(S, M, F, ray, ystage[i], nf, nu, &as[(size_t)i * nf], &es[(size_t)i * nf]);
            bool all_opaque = true;
            for (int k = 0; k < nf; ++k) {
                double ak[6], ek[6];
                for (int i = 0; i < 6; ++i) { ak[i] = as[(size_t)i * nf + k]; ek[i] = es[(size_t)i * nf + k]; }
                rt_rk_step(T, ak, ek, h_used, M.tau_max, &tau[k], &I[k]);
                if (!(tau[k] > M.tau_max)) all_opaque = false;
            }
            if (flag < 0 && all_opaque) flag = OPAQUE;
        }
        for (int v = 0; v < NV; ++v) y[v] = ynew[v];
        h = h_next;
        lambda += h_used;
        if (path) { path->nodes.insert(path->nodes.end(), y, y + 5); path->nodes.push_back(lambda); path->nodes.push_back(y[5]); if (nf > 0) path->absorb.push_back(a0[0]); }
    }
    out->flag = flag; out->r = y[0]; out->th = y[1]; out->ph = y[2] + phi_plane; out->t = y[5];   // (DISK: azimuth of the point on the plane)
    out->n_attempt = n_attempt; out->n_accept = n_accept;
    out->g = g; out->r_e = r_e;
    out->I = I; out->tau = tau;
}

inline void pixel_xy(const Scene& S, int i, int j, double* x, double* y) {   // step 1 [reading K]
    *x = S.x_min + (i + 0.5) * (S.x_max - S.x_min) / S.nx;
    *y = S.y_min + (j + 0.5) * (S.y_max - S.y_min) / S.ny;
}

// Step 12: thin-disk pixel value g^g_power r_e^-emis_index.
double disk_value(const Model& M, const RayOut& R) {
    if (R.flag != DISK || !(R.g > 0.0)) return 0.0;
    return std::pow(R.g, M.g_power) * std::pow(R.r_e, -M.emis_index);
}

// Kind 4 [reading NT of PAPER.md:L225-238, eq. (35)]: the relativistic multi-temperature disk of Novikov & Thorne
// (1973) / Page & Thorne (1974).  eq. (35): F(r) = 3 Mdot M f(r) / (8 pi r^3) = sigma T_eff^4; the paper does not
// print f(r) ("a correction factor related to the inner boundary of the disk and relativistic effects" that vanishes
// at r_isco).  It is Page & Thorne's closed form for zero torque at the marginally stable orbit, with x = sqrt(r),
// x0 = sqrt(r_isco) and x1, x2, x3 the roots of x^3 - 3x + 2a = 0:
//   f = x^2/(x^3 - 3x + 2a) [ x - x0 - (3/2) a ln(x/x0) - sum_i 3 (x_i - a)^2 / (x_i (x_i - x_j)(x_i - x_k)) ln((x - x_i)/(x0 - x_i)) ],
// which tends to 1 - ... -> 1 far out (the Newtonian 3 G M Mdot / 8 pi r^3).
double page_thorne_f(double a, double r) {
    const double r0 = isco_radius(a);
    if (!(r > r0)) return 0.0;
    const double x = std::sqrt(r), x0 = std::sqrt(r0);
    const double th = std::acos(a) / 3.0;
    const double x1 = 2.0 * std::cos(th - PI / 3.0), x2 = 2.0 * std::cos(th + PI / 3.0), x3 = -2.0 * std::cos(th);
    auto term = [&](double xi, double xj, double xk) {
        return 3.0 * (xi - a) * (xi - a) / (xi * (xi - xj) * (xi - xk)) * std::log((x - xi) / (x0 - xi));
    };
    const double br = x - x0 - 1.5 * a * std::log(x / x0) - term(x1, x2, x3) - term(x2, x1, x3) - term(x3, x1, x2);
    return x * x / (x * x * x - 3.0 * x + 2.0 * a) * br;
}

// T_eff(r) in kelvin from eq. (35) in cgs: F = 3 Mdot c^6 f / (8 pi G^2 M^2 r^3) with r in units of G M / c^2.
double nt_temperature(const Model& M, double a, double r) {
    const double Mg = GM_SUN * M.mbh_msun / G_NEWTON;                 // mass in grams
    const double c6 = std::pow(C_LIGHT, 6);
    const double F = 3.0 * M.mdot_gs * c6 * page_thorne_f(a, r) / (8.0 * PI * G_NEWTON * G_NEWTON * Mg * Mg * r * r * r);
    return (F > 0.0) ? std::pow(F / SIGMA_SB, 0.25) : 0.0;
}

// Observed specific intensity of the disk surface (blackbody at T_eff, no colour correction): the invariant
// I_nu / nu^3 is conserved, so I_nu(obs) = g^3 B_{nu/g}(T_eff(r_e)) = (2 h nu^3 / c^2) / expm1(h nu / (g k T_eff)).
double nt_intensity(const Scene& S, const Model& M, const RayOut& R, double nu) {
    if (R.flag != DISK || !(R.g > 0.0)) return 0.0;
    const double T = nt_temperature(M, S.a, R.r_e);
    if (!(T > 0.0)) return 0.0;
    const double xx = H_PLANCK * nu / (R.g * K_BOLTZ * T);
    return (2.0 * H_PLANCK * nu * nu * nu / (C_LIGHT * C_LIGHT)) / std::expm1(xx);
}

// Kind 3 [reading HS of PAPER.md:L252-264, eq. (36), Figs. 7, 8]: a hot spot on the opaque equatorial plane.
// Its centre moves on the prograde circular orbit of radius r_s with Omega_s = 1/(r_s^{3/2} + a),
// phi_s(t) = phi_0 + Omega_s t.  A ray that reaches the plane at (r_e, phi_e) after the coordinate time t_e
// (negative: the ray is traced backwards from the image plane, where t = 0) left it at t_em = t_obs + t_e; the
// surface brightness there is g^p exp(-d^2 / 2 r_spot^2) for d < 4 r_spot, d the distance to the spot centre
// at t_em in the pseudo-Cartesian coordinates of eqs. (33), (34), and 0 otherwise.
double hot_spot_value(const Scene& S, const Model& M, const RayOut& R, double t_obs) {
    if (R.flag != DISK || !(R.g > 0.0)) return 0.0;
    const double a = S.a;
    const double rs = (M.spot_r_orbit > 0.0) ? M.spot_r_orbit : isco_radius(a);
    const double Omega = 1.0 / (rs * std::sqrt(rs) + a);
    const double phi_s = M.spot_phi0 + Omega * (t_obs + R.t);
    const double Re = std::sqrt(R.r_e * R.r_e + a * a), Rs = std::sqrt(rs * rs + a * a);
    const double d2 = Re * Re + Rs * Rs - 2.0 * Re * Rs * std::cos(R.ph - phi_s);
    if (!(d2 < 16.0 * M.spot_size * M.spot_size)) return 0.0;
    return std::pow(R.g, M.g_power) * std::exp(-d2 / (2.0 * M.spot_size * M.spot_size));
}

}  // namespace

// ================================================================================================
// C interface for the tests (ctypes).  All pointers are host memory owned by the caller.
// ================================================================================================
extern "C" {

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

// out = {r_h, r_isco, E_isco, L_isco}
void oracle_kerr_constants(double a, double* out) {
    Flow F = make_flow(a);
    out[0] = horizon_radius(a); out[1] = F.r_isco; out[2] = F.E_isco; out[3] = F.L_isco;
}

// st = (r, theta, phi, p_r, p_theta); cons = {E, L, Q, E2_raw, L_raw}
void oracle_init_ray(const Scene* S, double x, double y, double* st, double* cons) {
    Ray ray; double raw[2]; double st6[NV];
    init_ray(*S, x, y, &ray, st6, raw);
    for (int v = 0; v < 5; ++v) st[v] = st6[v];
    cons[0] = ray.E; cons[1] = ray.L; cons[2] = ray.Q; cons[3] = raw[0]; cons[4] = raw[1];
}

// y[5] in, dy[6] out: (r, theta, phi, p_r, p_theta) and, last, dt/dlambda of eq. (9)
void oracle_rhs(double a, double E, double L, const double* y, double* dy) {
    Ray ray{a, E, L, 0.0};
    double y6[NV] = {y[0], y[1], y[2], y[3], y[4], 0.0};
    rhs(ray, y6, dy);
}

double oracle_null_ratio(double a, double E, double L, const double* y) {
    Ray ray{a, E, L, 0.0};
    return null_ratio(ray, y);
}

double oracle_carter_Q(double a, double E, double L, const double* y) {
    Ray ray{a, E, L, 0.0};
    return carter_Q(ray, y);
}

// c[6], A[36] row-major, b5[6], b4[6]
void oracle_tableau(int which, double* c, double* A, double* b5, double* b4) {
    Tableau T = make_tableau(which);
    std::memcpy(c, T.c, sizeof(T.c)); std::memcpy(A, T.A, sizeof(T.A));
    std::memcpy(b5, T.b5, sizeof(T.b5)); std::memcpy(b4, T.b4, sizeof(T.b4));
}

void oracle_rk_attempt(double a, double E, double L, int which, const double* y, double h, double* ynew, double* yerr) {
    Ray ray{a, E, L, 0.0};
    Tableau T = make_tableau(which);
    double y6[NV] = {y[0], y[1], y[2], y[3], y[4], 0.0}, yn[NV], ye[NV];
    rk_attempt(ray, T, y6, h, yn, ye);
    for (int v = 0; v < 5; ++v) { ynew[v] = yn[v]; yerr[v] = ye[v]; }
}

double oracle_error_norm(const double* y, const double* yerr, double rtol) {
    double y6[NV] = {y[0], y[1], y[2], y[3], y[4], 0.0}, e6[NV] = {yerr[0], yerr[1], yerr[2], yerr[3], yerr[4], 0.0};
    return error_norm(y6, e6, rtol);
}

// u[4] = (ut, ur, utheta, uphi); returns 1 if the flow has a velocity there; *gamma = eq. (2).
int oracle_flow_gamma(double a, double r, double th, double pr, double pth, double L, double* u, double* gamma) {
    Flow F = make_flow(a);
    if (!flow_velocity(a, F, r, th, u)) { *gamma = 0.0; return 0; }
    Ray ray{a, -1.0, L, 0.0};
    double y[NV] = {r, th, 0.0, pr, pth, 0.0};
    *gamma = gamma_shift(ray, y, u);
    return 1;
}

double oracle_bessel_K2(double x) { return bessel_K2(x); }
double oracle_mahadevan_M(double xM) { return mahadevan_M(xM); }
double oracle_planck_B(double nu, double T) { return planck_B(nu, T); }
double oracle_rg_cm(double mbh_msun) { return GM_SUN * mbh_msun / (C_LIGHT * C_LIGHT); }

// out = {n_e, T_e, B, Theta_e, nu_c, j, alpha}
void oracle_synchrotron(const Model* M, double a, double r, double th, double nu0, double* out) {
    Plasma p = plasma_state(*M, a, r, th);
    double j, al;
    synchrotron_coefficients(*M, p, nu0, &j, &al);
    out[0] = p.n_e; out[1] = p.T_e; out[2] = p.B; out[3] = p.Theta_e; out[4] = p.nu_c; out[5] = j; out[6] = al;
}

// state = {tau, T, I}, updated in place
void oracle_rt_update(double a0, double a1, double e0, double e1, double dl, double tau_max, double* state) {
    rt_update(a0, a1, e0, e1, dl, tau_max, &state[0], &state[1], &state[2]);
}

double oracle_page_thorne_f(double a, double r) { return page_thorne_f(a, r); }
double oracle_nt_temperature(const Model* M, double a, double r) { return nt_temperature(*M, a, r); }

// a[6], eps[6]: coefficients at the six stages; state = {tau, I}, updated in place [reading E']
void oracle_rt_rk_step(int which, const double* a, const double* eps, double h, double tau_max, double* state) {
    Tableau T = make_tableau(which);
    rt_rk_step(T, a, eps, h, tau_max, &state[0], &state[1]);
}

// Trace n rays that start at arbitrary image-plane points (xs[k], ys[k]).  Any output may be NULL.
// I and tau are [n][nf] (invariant intensity I_nu/nu^3, cgs / Hz^3).
void oracle_trace_points(const Scene* S, const Model* M, int nf, const double* nu, int n,
                         const double* xs, const double* ys,
                         int32_t* flag, double* r, double* th, double* ph,
                         int32_t* n_attempt, int32_t* n_accept,
                         double* g, double* r_e, double* I, double* tau, double* t) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < n; ++k) {
        RayOut R;
        trace_ray(*S, *M, nf, nu, xs[k], ys[k], &R, nullptr);
        if (flag) flag[k] = R.flag;
        if (r) r[k] = R.r;
        if (th) th[k] = R.th;
        if (ph) ph[k] = R.ph;
        if (n_attempt) n_attempt[k] = R.n_attempt;
        if (n_accept) n_accept[k] = R.n_accept;
        if (g) g[k] = R.g;
        if (r_e) r_e[k] = R.r_e;
        if (t) t[k] = R.t;
        for (int q = 0; q < nf; ++q) {
            if (I) I[(size_t)k * nf + q] = R.I[q];
            if (tau) tau[(size_t)k * nf + q] = R.tau[q];
        }
    }
}

// Accepted nodes of one ray: nodes[max_nodes][7] = (r, theta, phi, p_r, p_theta, lambda, t); returns the number of nodes (start included);
// cons = {E, L, Q}; res = {flag, n_attempt, n_accept}.
int oracle_trace_path(const Scene* S, const Model* M, double x, double y, int max_nodes, double* nodes,
                      double* cons, int32_t* res) {
    Ray ray; double st[NV];
    init_ray(*S, x, y, &ray, st, nullptr);
    cons[0] = ray.E; cons[1] = ray.L; cons[2] = ray.Q;
    RayOut R; Path P;
    trace_ray(*S, *M, 0, nullptr, x, y, &R, &P);
    int n = (int)(P.nodes.size() / 7);
    int m = std::min(n, max_nodes);
    std::memcpy(nodes, P.nodes.data(), sizeof(double) * 7 * (size_t)m);
    res[0] = R.flag; res[1] = R.n_attempt; res[2] = R.n_accept;
    return n;
}

// The same with the transfer at one frequency along the ray (kind 2): absorb[n] = the invariant absorption
// coefficient at each node (what the Δτ cap of reading DT looks at); res = {flag, n_attempt, n_accept}.
int oracle_trace_path_rt(const Scene* S, const Model* M, double nu_hz, double x, double y, int max_nodes,
                         double* nodes, double* absorb, int32_t* res) {
    RayOut R; Path P;
    trace_ray(*S, *M, 1, &nu_hz, x, y, &R, &P);
    int n = (int)(P.nodes.size() / 7);
    int m = std::min(n, max_nodes);
    std::memcpy(nodes, P.nodes.data(), sizeof(double) * 7 * (size_t)m);
    for (int k = 0; k < m && k < (int)P.absorb.size(); ++k) absorb[k] = P.absorb[k];
    res[0] = R.flag; res[1] = R.n_attempt; res[2] = R.n_accept;
    return n;
}

// --- the three image drivers; the CUDA library's entry points compute the same outputs ----------
// Pixels are either the whole grid (idx_i == NULL: n = nx*ny, row-major [j][i]) or the listed ones.

// Geodesics only (C0).
void oracle_trace_geodesics(const Scene* S, int n, const int32_t* idx_i, const int32_t* idx_j,
                            int32_t* flag, double* r, double* th, double* ph,
                            int32_t* n_attempt, int32_t* n_accept, double* t) {
    Model M; std::memset(&M, 0, sizeof(M));
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < n; ++k) {
        int i = idx_i ? idx_i[k] : k % S->nx, j = idx_j ? idx_j[k] : k / S->nx;
        double x, y; pixel_xy(*S, i, j, &x, &y);
        RayOut R;
        trace_ray(*S, M, 0, nullptr, x, y, &R, nullptr);
        flag[k] = R.flag; r[k] = R.r; th[k] = R.th; ph[k] = R.ph;
        n_attempt[k] = R.n_attempt; n_accept[k] = R.n_accept;
        if (t) t[k] = R.t;
    }
}

// One frequency (C1, C2, C4).  kind 1: image = g^p r_e^-q, aux0 = g, aux1 = r_e, hist[nbins] over g
// (only when the whole grid is rendered).  kind 2: image = I_nu = nu^3 * invariant intensity (cgs),
// aux0 = tau, aux1 = 0.
void oracle_render_image(const Scene* S, const Model* M, double nu_hz, int n, const int32_t* idx_i, const int32_t* idx_j,
                         double* image, double* aux0, double* aux1, int32_t* flag, int32_t* n_attempt,
                         int32_t* n_accept, double* hist) {
    int nf = (M->kind == 2) ? 1 : 0;
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < n; ++k) {
        int i = idx_i ? idx_i[k] : k % S->nx, j = idx_j ? idx_j[k] : k / S->nx;
        double x, y; pixel_xy(*S, i, j, &x, &y);
        RayOut R;
        trace_ray(*S, *M, nf, &nu_hz, x, y, &R, nullptr);
        if (M->kind == 1) { image[k] = disk_value(*M, R); aux0[k] = R.g; aux1[k] = R.r_e; }
        else if (M->kind == 2) { image[k] = nu_hz * nu_hz * nu_hz * R.I[0]; aux0[k] = R.tau[0]; aux1[k] = 0.0; }
        else { image[k] = 0.0; aux0[k] = 0.0; aux1[k] = 0.0; }
        flag[k] = R.flag; n_attempt[k] = R.n_attempt;
        if (n_accept) n_accept[k] = R.n_accept;
    }
    if (hist && M->kind == 1 && M->nbins > 0) {       // serial, pixel order: line profile [reading Q]
        double area = ((S->x_max - S->x_min) / S->nx) * ((S->y_max - S->y_min) / S->ny);
        for (int b = 0; b < M->nbins; ++b) hist[b] = 0.0;
        for (int k = 0; k < n; ++k) {
            if (flag[k] != DISK) continue;
            double g = aux0[k];
            if (!(g >= M->g_lo && g < M->g_hi)) continue;
            int b = (int)std::floor((g - M->g_lo) / (M->g_hi - M->g_lo) * M->nbins);
            if (b >= M->nbins) b = M->nbins - 1;
            hist[b] += image[k] * area;
        }
    }
}

// Hot spot (kind 3): images [nt][n], lightcurve[nt] = sum(image) * pixel area, spectrogram [nt][nbins] over g
// (only when the whole grid is rendered); per pixel g, r_e, phi_e, t_e of the disk crossing.
void oracle_render_hotspot(const Scene* S, const Model* M, const double* t_obs, int nt, int n,
                           const int32_t* idx_i, const int32_t* idx_j,
                           double* images, double* lightcurve, double* spectrogram,
                           double* g, double* r_e, double* phi_e, double* t_e, int32_t* flag, int32_t* n_attempt) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < n; ++k) {
        int i = idx_i ? idx_i[k] : k % S->nx, j = idx_j ? idx_j[k] : k / S->nx;
        double x, y; pixel_xy(*S, i, j, &x, &y);
        RayOut R;
        trace_ray(*S, *M, 0, nullptr, x, y, &R, nullptr);
        for (int q = 0; q < nt; ++q) images[(size_t)q * n + k] = hot_spot_value(*S, *M, R, t_obs[q]);
        bool hit = (R.flag == DISK);
        g[k] = R.g; r_e[k] = R.r_e; phi_e[k] = hit ? R.ph : 0.0; t_e[k] = hit ? R.t : 0.0;
        flag[k] = R.flag; n_attempt[k] = R.n_attempt;
    }
    double area = ((S->x_max - S->x_min) / S->nx) * ((S->y_max - S->y_min) / S->ny);
    for (int q = 0; q < nt; ++q) {
        double sum = 0.0;
        for (int k = 0; k < n; ++k) sum += images[(size_t)q * n + k];
        if (lightcurve) lightcurve[q] = sum * area;
        if (spectrogram && M->nbins > 0) {
            double* h = spectrogram + (size_t)q * M->nbins;
            for (int b = 0; b < M->nbins; ++b) h[b] = 0.0;
            for (int k = 0; k < n; ++k) {
                double v = images[(size_t)q * n + k];
                if (v == 0.0 || !(g[k] >= M->g_lo && g[k] < M->g_hi)) continue;
                int b = (int)std::floor((g[k] - M->g_lo) / (M->g_hi - M->g_lo) * M->nbins);
                if (b >= M->nbins) b = M->nbins - 1;
                h[b] += v * area;
            }
        }
    }
}

// nf frequencies at once (C3): images [nf][n] = I_nu (cgs); nuLnu[nf] = 4 pi nu r_g^2 dx dy sum I_nu
// (erg/s, step 13; only meaningful when the whole grid is rendered).
void oracle_render_spectrum(const Scene* S, const Model* M, const double* nu_hz, int nf, int n,
                            const int32_t* idx_i, const int32_t* idx_j,
                            double* images, double* nuLnu, int32_t* flag, int32_t* n_attempt) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < n; ++k) {
        int i = idx_i ? idx_i[k] : k % S->nx, j = idx_j ? idx_j[k] : k / S->nx;
        double x, y; pixel_xy(*S, i, j, &x, &y);
        RayOut R;
        if (M->kind == 4) {                      // Novikov-Thorne disk: evaluated at the crossing, no transfer along the ray
            trace_ray(*S, *M, 0, nullptr, x, y, &R, nullptr);
            for (int q = 0; q < nf; ++q) images[(size_t)q * n + k] = nt_intensity(*S, *M, R, nu_hz[q]);
            if (flag) flag[k] = R.flag;
            if (n_attempt) n_attempt[k] = R.n_attempt;
            continue;
        }
        trace_ray(*S, *M, nf, nu_hz, x, y, &R, nullptr);
        for (int q = 0; q < nf; ++q) images[(size_t)q * n + k] = nu_hz[q] * nu_hz[q] * nu_hz[q] * R.I[q];
        if (flag) flag[k] = R.flag;
        if (n_attempt) n_attempt[k] = R.n_attempt;
    }
    if (nuLnu) {
        double rg = GM_SUN * M->mbh_msun / (C_LIGHT * C_LIGHT);
        double area = ((S->x_max - S->x_min) / S->nx) * ((S->y_max - S->y_min) / S->ny);
        for (int q = 0; q < nf; ++q) {
            double sum = 0.0;
            for (int k = 0; k < n; ++k) sum += images[(size_t)q * n + k];
            nuLnu[q] = 4.0 * PI * nu_hz[q] * rg * rg * area * sum;
        }
    }
}

}  // extern "C"
