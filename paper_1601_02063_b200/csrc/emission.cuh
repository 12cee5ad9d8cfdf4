// emission.cuh — device-side flow, energy shift and thermal-synchrotron coefficients.
//
//   flow_igamma    : flow four-velocity (Keplerian shells with u^θ = 0 outside the ISCO, PAPER.md:L268;
//                    plunging with the ISCO's E, L inside, BASELINE.json:configs[2]) and 1/γ, γ the
//                    energy-shift factor of eq. (2).
//   bessel_k2_inv  : 1/K_2(x) of eq. (37) as (factor, exponent); tables from gen_bessel_k2.py.
//   rt_point       : plasma state (BASELINE.json:configs[2]) and everything the frequencies share.
//   rt_coefficients: per-frequency a = r_g α_0(ν_0)/γ and ε = r_g j_0(ν_0)/(γ ν_0³) of eqs. (30), (31)
//                    with eqs. (37)-(39) and Kirchhoff's law.
//   rt_update      : one accepted step of eqs. (30), (31) (reading E).
//
// Arithmetic layout.  Every factor of ε is a power law or an exponential, so the
// product is assembled in log space and exponentiated ONCE per frequency:
//   ε = r_g j_coef ν_0 n_e M(x_M) / (K_2(1/Θ_e) γ ν_0³)
//     = r_g · Kfac · u² (1 + 0.40 u³ + 0.5316 u⁶) · exp( E + c_k − 1.8899 t⁴ ),
//   t = x_M^(1/12) = ν_k^(1/12) · exp((ln(1/γ) − ln ν_c)/12),  u = 1/t,   (eq. (38): x^1/6 = t², x^1/4 = t³, x^1/3 = t⁴)
//   E = ln(4.0505 j_coef) + ln n_e + Kexp − ln(1/γ),  c_k = −2 ln ν_k,  1/K_2 = Kfac · e^Kexp,
//   a = ε · expm1(h ν_0 / k T_e) · c²/(2h)                              (Kirchhoff with B_ν0(T_e)),
// with ln n_e, ln Θ_e, ln ν_c linear in ln r, cos²θ and constants.  Per point this needs two logarithms
// (ln r, ln 1/γ) and two exponentials (1/Θ_e, t/ν^(1/12)); per frequency one exponential and one expm1, instead of
// the dozen pow/exp/cbrt/sqrt/divisions of the formulas as printed.  Same mathematics, different
// rounding (parity tolerance on images: 1e-6 relative L1).
#pragma once
#include "params.h"
#include "dmath.cuh"
#include "bessel_k2_coeffs.h"

namespace ody {

// 1/γ = u^t + p_r u^r + L u^φ for k_t = −E = 1 (eq. (2) with a static observer at infinity).
// s, c = sinθ, cosθ.  Returns false where the flow has no normalisable velocity.
__device__ __forceinline__ bool flow_igamma(const Params& P, const double L, const double r, const double s, const double c,
                                            const double pr, double& igam) {
    const double a = P.a, a2 = P.a2;
    const double s2 = s * s, r2 = r * r;
    const double Sigma = fma(a2, c * c, r2);
    const double Delta = fma(r, r - 2.0, a2);
    const double iS = d_rcp(Sigma);
    // covariant metric, eq. (1)
    const double g_tt = -(1.0 - 2.0 * r * iS);
    const double g_tp = -2.0 * a * r * s2 * iS;
    const double g_pp = (r2 + a2 + 2.0 * a2 * r * s2 * iS) * s2;
    double Omega, ur = 0.0, ur2_grr = 0.0;
    if (r >= P.r_isco) {
        Omega = d_rcp(fma(r, d_sqrt(r), a));
    } else {
        const double E = P.E_isco, Lk = P.L_isco, ir = d_rcp(r);
        const double ut_eq = (r2 + a2 + 2.0 * a2 * ir) * E - 2.0 * a * ir * Lk;      // × 1/Δ, cancels in Ω
        const double up_eq = 2.0 * a * ir * E + (1.0 - 2.0 * ir) * Lk;
        Omega = up_eq * d_rcp(ut_eq);
        const double dl = Lk - a * E;
        double ur2 = E * E - 1.0 + 2.0 * ir - (Lk * Lk - a2 * (E * E - 1.0)) * ir * ir + 2.0 * dl * dl * ir * ir * ir;
        if (ur2 > 0.0) {
            ur = -d_sqrt(ur2);
            ur2_grr = ur2 * Sigma * d_rcp(Delta);                                 // g_rr (u^r)²
        }
    }
    const double N = -(g_tt + 2.0 * Omega * g_tp + Omega * Omega * g_pp);
    if (!(N > 0.0)) return false;
    double ut = d_rsqrt(N);
    if (ur2_grr > 0.0) ut *= d_sqrt(1.0 + ur2_grr);                              // plunging region only
    igam = fma(ut, fma(L, Omega, 1.0), pr * ur);
    return true;
}

// PREC = 0: FP64 throughout.  PREC = 1: the mixed-precision variant of north_star subsystem (c) — exponent sums,
// argument reductions and accumulators stay FP64, the polynomial cores of exp / expm1 / log and the K_2
// polynomials run in FP32.
template <int PREC> __device__ __forceinline__ double p_exp_nc(double x) { return PREC ? f_exp_nc(x) : d_exp_nc(x); }
template <int PREC> __device__ __forceinline__ double p_exp(double x) { return PREC ? f_exp(x) : d_exp(x); }
template <int PREC> __device__ __forceinline__ double p_expm1_nc(double x) { return PREC ? f_expm1_nc(x) : d_expm1_nc(x); }
template <int PREC> __device__ __forceinline__ double p_log(double x) { return PREC ? f_log(x) : d_log(x); }

#define ODY_X(i, v) v,
#define ODY_XF(i, v) (float)(v),
__constant__ float kK2Af[ODY_K2_NS] = { ODY_K2_A(ODY_XF) };
__constant__ float kK2Bf[ODY_K2_NS] = { ODY_K2_B(ODY_XF) };
__constant__ float kK2Pf[ODY_K2_NC + 1] = { ODY_K2_P(ODY_XF) };
#undef ODY_XF
__constant__ double kK2A[ODY_K2_NS] = { ODY_K2_A(ODY_X) };
__constant__ double kK2B[ODY_K2_NS] = { ODY_K2_B(ODY_X) };
__constant__ double kK2P[ODY_K2_NC + 1] = { ODY_K2_P(ODY_X) };
#undef ODY_X
// 1/K_2(x) = kfac · exp(kexp) for 0 < x; lx = ln x.
template <int PREC>
__device__ __forceinline__ void bessel_k2_inv(const double x, const double lx, double& kfac, double& kexp) {
    if (PREC == 1) {                                                  // same formulas, Horner chains in FP32
        const float t = (float)(0.25 * x * x), z = (float)fma(4.0, d_rcp(x), -1.0);
        float A = 0.0f, B = 0.0f, F = 0.0f;
#pragma unroll
        for (int k = ODY_K2_NS - 1; k >= 0; --k) { A = fmaf(A, t, kK2Af[k]); B = fmaf(B, t, kK2Bf[k]); }
#pragma unroll
        for (int k = ODY_K2_NC; k >= 0; --k) F = fmaf(F, z, kK2Pf[k]);
        const double lg = lx - 0.69314718055994530942;
        const double td = 0.25 * x * x;
        const double S = fma(4.0 * td * td, fma(-lg, (double)A, (double)B), fma(-2.0, td, 2.0));
        const bool small = x <= 2.0;
        kfac = d_rcp(small ? S : (double)F);
        kexp = small ? 2.0 * lx : x + fma(0.5, lx, -0.22579135264472743236);
        return;
    }
    // Both representations are evaluated and one is selected: in a warp whose lanes sit on both sides of
    // x = 2 a branch would execute both bodies anyway, one after the other; straight-line code lets the two
    // (independent) Horner chains interleave.  Neither overflows on the other's domain (x < 700).
    const double* const ca = kK2A; const double* const cb = kK2B; const double* const cp = kK2P;
    const double t = 0.25 * x * x;
    const double z = fma(4.0, d_rcp(x), -1.0);
    double A = 0.0, B = 0.0, F = 0.0;
#pragma unroll
    for (int k = ODY_K2_NS - 1; k >= 0; --k) { A = fma(A, t, ca[k]); B = fma(B, t, cb[k]); }
#pragma unroll
    for (int k = ODY_K2_NC; k >= 0; --k) F = fma(F, z, cp[k]);
    const double lg = lx - 0.69314718055994530942;                   // ln(x/2)
    // x <= 2:  x² K_2 = 2 − 2t + 4t² (B − ln(x/2) A)          ->  1/K_2 = x² / S
    // x >  2:  K_2 = sqrt(π/2x) e^−x F(z)                       ->  1/K_2 = e^{x + ½ ln x + ½ ln(2/π)} / F
    const double S = fma(4.0 * t * t, fma(-lg, A, B), fma(-2.0, t, 2.0));
    const bool small = x <= 2.0;
    kfac = d_rcp(small ? S : F);
    kexp = small ? 2.0 * lx : x + fma(0.5, lx, -0.22579135264472743236);
}

// What all frequencies share at one point of the ray.
struct RtPoint {
    bool on;            // inside the emitting region with a valid flow
    double fac;         // r_g · Kfac
    double E;           // exponent shared by all frequencies
    double t0, u0;      // spectrum kernel: (x_M / ν)^(1/12) and its reciprocal, x_M^(1/12) = t0 ν^(1/12)
    double lxm0;        // single-frequency kernels: ln(x_M / ν) = ln(1/γ) − ln ν_c
    double ycoef;       // h ν_0 /(k T_e) = ν · ycoef
};

// HOIST: evaluate the x_M^(1/12) exponential once per point (spectrum kernel: ν_k^(1/12) is a constant per
// frequency) instead of once per frequency (single-frequency kernels: same work, fewer live registers).
template <bool HOIST, int PREC = 0>
__device__ __forceinline__ void rt_point(const Params& P, const double L, const double r, const double s, const double c,
                                         const double pr, RtPoint& q) {
    q.on = false; q.fac = 0.0; q.E = 0.0; q.t0 = 1.0; q.u0 = 1.0; q.lxm0 = 0.0; q.ycoef = 0.0;   // off: every coefficient evaluates to 0
    if (!(r > P.r_cap && r < P.r_rt_out)) return;
    double igam;
    if (!flow_igamma(P, L, r, s, c, pr, igam)) return;
    if (!(igam > 0.0) || isinf(igam)) return;
    const double lr = p_log<PREC>(r);
    const double lrel = lr - P.ln_rh;                               // ln(r / r_h)
    const double ln_ne = fma(P.n_index, lrel, fma(-c * c, P.inv_2h2, P.ln_n0));
    const double ln_Th = fma(P.T_index, lrel, P.ln_Theta0);         // ln Θ_e
    if (!(ln_Th > -6.5 && ln_Th < 690.0)) return;                   // 1/Θ_e > 665: K_2 underflows, no emission
    if (!(ln_ne > -1e300)) return;                                  // n0 = 0
    const double x = p_exp_nc<PREC>(-ln_Th);                        // 1/Θ_e
    double kfac, kexp;
    bessel_k2_inv<PREC>(x, -ln_Th, kfac, kexp);
    const double ligam = p_log<PREC>(igam);
    // ln ν_c = ln nuc_coef + ½ (ln B2_coef + ln n_e − ln r) + 2 ln Θ_e         (eq. (39), B² = B2_coef n_e / r)
    const double ln_nuc = fma(0.5, ln_ne - lr, fma(2.0, ln_Th, P.ln_nuc0));
    q.on = true;
    q.fac = P.rg_cm * kfac;
    q.E = P.ln_j0 + ln_ne + kexp - ligam;
    if (HOIST) {
        q.t0 = p_exp_nc<PREC>((ligam - ln_nuc) * (1.0 / 12.0));     // ln(x_M/ν) = ln(1/γ) − ln ν_c; |argument| < 700
        q.u0 = d_rcp(q.t0);
    } else {
        q.lxm0 = ligam - ln_nuc;
    }
    q.ycoef = P.h_over_mc2 * igam * x;
}

// Per-frequency coefficients.  ln_nu = ln ν_k.
// Per-frequency constants.  The fused kernels index the Params tables with a warp-uniform k (uniform
// constant loads); the two-phase spectrum kernel, where k is the LANE's frequency, must fetch them once into
// registers — a constant load with 32 different addresses is replayed 32 times.
struct Freq { double nu, ln_nu, nu12, inu12; };
__device__ __forceinline__ Freq freq_of(const Params& P, const int k) { return Freq{P.nu[k], P.ln_nu[k], P.nu12[k], P.inu12[k]}; }

template <bool HOIST, int PREC = 0>
__device__ __forceinline__ void rt_coefficients(const Params& P, const RtPoint& q, const Freq& f, double& acoef, double& ecoef) {
    const double nu = f.nu, ln_nu = f.ln_nu;
    // straight-line on purpose (no early return when the point is off: fac = 0 gives ε = a = 0), so that the
    // spectrum kernel's unrolled frequency loop can interleave independent chains
    double t, u;                                                     // x_M^(1/12) and its reciprocal
    if (HOIST) { t = q.t0 * f.nu12; u = q.u0 * f.inu12; }
    else { t = d_exp_nc((ln_nu + q.lxm0) * (1.0 / 12.0)); u = d_rcp(t); }   // FP64 in both variants: t^4 sits in an exponent
    const double t2 = t * t, u2 = u * u;
    const double u3 = u2 * u;
    const double poly = fma(u3, fma(0.5316, u3, 0.40), 1.0);        // eq. (38) bracket
    const double ex = p_exp<PREC>(fma(-1.8899, t2 * t2, fma(-2.0, ln_nu, q.E)));
    const double eps = q.fac * u2 * poly * ex;                       // reading D, F
    const double ya = nu * q.ycoef;                                  // hν0/kT_e >= 0
    const bool planck_ok = ya < 700.0;                               // beyond: B_ν underflows, α = 0 as in the formula
    const double em1 = p_expm1_nc<PREC>(planck_ok ? ya : 700.0);     // e^{hν0/kT} − 1
    ecoef = eps;
    acoef = (eps > 0.0 && planck_ok) ? eps * em1 * P.inv_planck : 0.0;   // Kirchhoff
}

// Trapezoid in λ for Δτ and the emission, exact attenuation across the step: φ(x) = (1 − e^−x)/x.
template <int PREC = 0>
__device__ __forceinline__ void rt_update(const double a0, const double a1, const double e0, const double e1,
                                          const double dl, const double tau_max, double& tau, double& T, double& I) {
    const bool live = !(tau > tau_max);                              // a frozen frequency keeps its values (selects, no branch)
    const double dtau = 0.5 * (a0 + a1) * dl;
    const double em = p_expm1_nc<PREC>(dtau < 700.0 ? -dtau : -700.0);   // e^−Δτ − 1 (Δτ >= 0)
    const double phi = (dtau > 1e-300) ? -em * d_rcp(dtau) : 1.0;
    const double In = fma(T * (0.5 * (e0 + e1) * dl), phi, I);
    const double Tn = fma(T, em, T);
    I = live ? In : I;
    T = live ? Tn : T;
    tau = live ? tau + dtau : tau;
}

// The same update in two parts, for the transfer FIFO of the single-frequency kernel: what depends only on the
// coefficients at the two ends of the step (the expensive part: an exponential and a reciprocal), and the
// recurrence in tau, T, I.  Operation for operation the arithmetic of rt_update().
template <int PREC = 0>
__device__ __forceinline__ void rt_increments(const double a0, const double a1, const double e0, const double e1, const double dl,
                                              double& dtau, double& em, double& phi, double& w) {
    dtau = 0.5 * (a0 + a1) * dl;
    em = p_expm1_nc<PREC>(dtau < 700.0 ? -dtau : -700.0);
    phi = (dtau > 1e-300) ? -em * d_rcp(dtau) : 1.0;
    w = 0.5 * (e0 + e1) * dl;
}
__device__ __forceinline__ void rt_accumulate(const double dtau, const double em, const double phi, const double w,
                                              const double tau_max, double& tau, double& T, double& I) {
    const bool live = !(tau > tau_max);
    const double In = fma(T * w, phi, I);
    const double Tn = fma(T, em, T);
    I = live ? In : I;
    T = live ? Tn : T;
    tau = live ? tau + dtau : tau;
}

// ------------------------------------------------------------------------------------------------
// Novikov–Thorne disk (kind 4; eq. (35); reading NT): effective temperature at radius r,
// σ T_eff⁴ = 3 Mdot M f(r)/(8π r³) with Page & Thorne's closed form of f for zero torque at r_isco,
//   f = x²/(x³ - 3x + 2a) [x - x0 - (3/2) a ln(x/x0) - Σ_i c_i ln((x - x_i)/(x0 - x_i))],  x = sqrt(r).
// Evaluated once per ray (at its disk crossing), so the library's log/pow are used as they are.
__device__ __forceinline__ double nt_temperature(const Params& P, double r) {
    if (!(r > P.r_isco)) return 0.0;
    const double x = sqrt(r), x0 = P.nt_x0;
    double br = x - x0 - 1.5 * P.a * log(x / x0);
#pragma unroll
    for (int i = 0; i < 3; ++i) br -= P.nt_c[i] * log((x - P.nt_x[i]) / (x0 - P.nt_x[i]));
    const double f = x * x / (x * x * x - 3.0 * x + 2.0 * P.a) * br;
    const double T4 = P.nt_T4 * f / (r * r * r);
    return (T4 > 0.0) ? sqrt(sqrt(T4)) : 0.0;
}

}  // namespace ody
