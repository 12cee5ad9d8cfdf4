// emission.cuh — device-side flow, energy shift and thermal-synchrotron coefficients.
//
//   flow_gamma     : flow four-velocity (Keplerian shells with u^θ = 0 outside the ISCO, PAPER.md:L268;
//                    plunging with the ISCO's E, L inside, BASELINE.json:configs[2]) and the
//                    energy-shift factor γ of eq. (2).
//   bessel_k2      : K_2(x) of eq. (37); tables from gen_bessel_k2.py.
//   rt_point       : plasma state (BASELINE.json:configs[2]) and what every frequency shares.
//   rt_coefficients: per-frequency a = r_g α_0(ν_0)/γ and ε = r_g j_0(ν_0)/(γ ν_0³) of eqs. (30), (31)
//                    with eqs. (37)-(39) and Kirchhoff's law.
//   rt_update      : one accepted step of eqs. (30), (31) (reading E).
#pragma once
#include "params.h"
#include "bessel_k2_coeffs.h"

namespace ody {

// γ = 1/(u^t + p_r u^r + L u^φ) for k_t = −E = 1 (eq. (2) with a static observer at infinity).
// s, c = sinθ, cosθ.  Returns false where the flow has no normalisable velocity.
__device__ __forceinline__ bool flow_gamma(const Params& P, const double L, const double r, const double s, const double c,
                                           const double pr, double& gam) {
    const double a = P.a, a2 = P.a2;
    const double s2 = s * s, r2 = r * r;
    const double Sigma = fma(a2, c * c, r2);
    const double Delta = fma(r, r - 2.0, a2);
    const double iS = 1.0 / Sigma;
    // covariant metric, eq. (1)
    const double g_tt = -(1.0 - 2.0 * r * iS);
    const double g_tp = -2.0 * a * r * s2 * iS;
    const double g_pp = (r2 + a2 + 2.0 * a2 * r * s2 * iS) * s2;
    double Omega, ur = 0.0, ur2_grr = 0.0;
    if (r >= P.r_isco) {
        Omega = 1.0 / fma(r, sqrt(r), a);
    } else {
        const double E = P.E_isco, Lk = P.L_isco, ir = 1.0 / r;
        const double ut_eq = (r2 + a2 + 2.0 * a2 * ir) * E - 2.0 * a * ir * Lk;      // × 1/Δ, cancels in Ω
        const double up_eq = 2.0 * a * ir * E + (1.0 - 2.0 * ir) * Lk;
        Omega = up_eq / ut_eq;
        const double dl = Lk - a * E;
        double ur2 = E * E - 1.0 + 2.0 * ir - (Lk * Lk - a2 * (E * E - 1.0)) * ir * ir + 2.0 * dl * dl * ir * ir * ir;
        if (ur2 < 0.0) ur2 = 0.0;
        ur = -sqrt(ur2);
        ur2_grr = ur2 * Sigma / Delta;                                            // g_rr (u^r)²
    }
    const double N = -(g_tt + 2.0 * Omega * g_tp + Omega * Omega * g_pp);
    if (!(N > 0.0)) return false;
    const double ut = sqrt((1.0 + ur2_grr) / N);
    gam = 1.0 / (ut + pr * ur + L * Omega * ut);
    return true;
}

#define ODY_X(i, v) v,
__device__ __forceinline__ double bessel_k2(const double x) {
    if (x <= 2.0) {
        const double ca[ODY_K2_NS] = { ODY_K2_A(ODY_X) };
        const double cb[ODY_K2_NS] = { ODY_K2_B(ODY_X) };
        const double t = 0.25 * x * x;
        double A = 0.0, B = 0.0;
#pragma unroll
        for (int k = ODY_K2_NS - 1; k >= 0; --k) { A = fma(A, t, ca[k]); B = fma(B, t, cb[k]); }
        return 2.0 / (x * x) - 0.5 + t * (B - log(0.5 * x) * A);
    } else {
        const double cp[ODY_K2_NC + 1] = { ODY_K2_P(ODY_X) };
        const double z = 4.0 / x - 1.0;
        double F = 0.0;
#pragma unroll
        for (int k = ODY_K2_NC; k >= 0; --k) F = fma(F, z, cp[k]);
        return sqrt(1.5707963267948966 / x) * exp(-x) * F;
    }
}
#undef ODY_X

// What all frequencies share at one point of the ray.
struct RtPoint {
    bool on;            // inside the emitting region with a valid flow
    double gam;         // γ
    double n_e, T_e;    // cm^-3, K
    double nu_c;        // eq. (39)
    double jK;          // j_coef n_e / K_2(1/Θ_e)   (0 when K_2 underflows)
};

__device__ __forceinline__ void rt_point(const Params& P, const double L, const double r, const double s, const double c,
                                         const double pr, RtPoint& q) {
    q.on = false;
    if (!(r > P.r_cap && r < P.r_rt_out)) return;
    double gam;
    if (!flow_gamma(P, L, r, s, c, pr, gam)) return;
    if (!(gam > 0.0) || isinf(gam)) return;
    const double lx = log(r / P.r_h);
    const double n_e = P.n0 * exp(fma(P.n_index, lx, -c * c * P.inv_2h2));
    const double T_e = P.T0 * exp(P.T_index * lx);
    const double B = sqrt(P.B2_coef * n_e / r);
    const double Theta = P.theta_per_K * T_e;
    const double K2 = bessel_k2(1.0 / Theta);
    q.on = true; q.gam = gam; q.n_e = n_e; q.T_e = T_e;
    q.nu_c = P.nuc_coef * B * Theta * Theta;
    q.jK = (K2 > 0.0) ? P.j_coef * n_e / K2 : 0.0;
}

// eq. (38)
__device__ __forceinline__ double mahadevan_M(const double xM) {
    const double sq = sqrt(xM);          // x^1/2
    const double qq = sqrt(sq);          // x^1/4
    const double cb = cbrt(xM);          // x^1/3
    const double sx = sqrt(cb);          // x^1/6
    return 4.0505 / sx * (1.0 + 0.40 / qq + 0.5316 / sq) * exp(-1.8899 * cb);
}

__device__ __forceinline__ void rt_coefficients(const Params& P, const RtPoint& q, const double nu, double& acoef, double& ecoef) {
    acoef = 0.0; ecoef = 0.0;
    if (!q.on) return;
    const double igam = 1.0 / q.gam;
    const double nu0 = nu * igam;                                   // local frequency (reading D)
    const double Mx = mahadevan_M(nu0 / q.nu_c);
    const double j = (Mx > 0.0) ? q.jK * nu0 * Mx : 0.0;            // eq. (37) per steradian (reading F)
    const double nu03 = nu0 * nu0 * nu0;
    const double Bnu = P.planck_coef * nu03 / expm1(P.h_over_k * nu0 / q.T_e);
    const double alpha = (j > 0.0 && Bnu > 0.0) ? j / Bnu : 0.0;    // Kirchhoff
    acoef = P.rg_cm * alpha * igam;
    ecoef = P.rg_cm * j * igam / nu03;
}

// Trapezoid in λ for Δτ and the emission, exact attenuation across the step: φ(x) = (1 − e^−x)/x.
__device__ __forceinline__ void rt_update(const double a0, const double a1, const double e0, const double e1,
                                          const double dl, const double tau_max, double& tau, double& T, double& I) {
    if (tau > tau_max) return;
    const double dtau = 0.5 * (a0 + a1) * dl;
    const double em = expm1(-dtau);                                 // e^−Δτ − 1
    const double phi = (dtau > 0.0) ? -em / dtau : 1.0;
    I = fma(T * (0.5 * (e0 + e1) * dl), phi, I);
    T *= (1.0 + em);
    tau += dtau;
}

}  // namespace ody
