// geodesic.cuh — device-side Kerr null-geodesic arithmetic of the Odyssey hot path.
//
//   init_ray      : pixel -> Boyer–Lindquist state and constants of motion, §2.2,
//                   eqs. (18)-(26), (7), (8), (4), (5).
//   geodesic_rhs  : the five right-hand sides, eqs. (4), (5), (12) and -dH/dr, -dH/dθ of the
//                   un-substituted Hamiltonian (≡ eqs. (14), (15) on the null shell; DESIGN.md
//                   reading A), pole clamp of PAPER.md:L90.
//   rk_stages     : stages 2..6 of an embedded 6-stage Runge–Kutta 5(4) pair ("fifth-
//                   order Runge–Kutta … adaptive step size", Press et al. 1992) with the first
//                   slope k1 supplied by the caller (it is cached across rejected attempts).
//
// Photon energy is normalised to E = -1 (ray traced backwards in time; readings B, C),
// which is folded into the formulas below: P = (r²+a²)E − aL = −Pm with Pm = r² + a² + aL.
#pragma once
#include "params.h"

namespace ody {

struct State { double r, th, ph, pr, pth; };     // y of PAPER.md:L88 without t
struct Slope { double r, th, ph, pr, pth; };     // dy/dλ

// ------------------------------------------------------------------------------------------------
// Right-hand side.  Also returns sinθ, cosθ (unclamped) for the emission code.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void geodesic_rhs(const double a, const double a2, const double L,
                                             const double r, const double th, const double pr, const double pth,
                                             Slope& k, double& sin_th, double& cos_th) {
    double s, c;
    sincos(th, &s, &c);
    sin_th = s; cos_th = c;
    if (fabs(s) < 1e-8) s = copysign(1e-8, s);
    const double r2 = r * r;
    const double Sigma = fma(a2, c * c, r2);                      // Σ = r² + a² cos²θ
    const double Delta = fma(r, r - 2.0, a2);                     // Δ = r² − 2r + a²
    const double Pm = r2 + fma(a, L, a2);                         // −P
    const double iS = 1.0 / Sigma, iD = 1.0 / Delta, is = 1.0 / s;
    const double is2 = is * is;
    const double D = fma(L, is, a * s);                           // L/sinθ − aE sinθ
    const double q = Pm * iD;                                     // −P/Δ
    const double pr2 = pr * pr;
    const double G = fma(Delta, pr2, fma(pth, pth, fma(D, D, -Pm * q)));   // 2ΣH
    const double GiS = G * iS;
    k.r = Delta * pr * iS;                                        // eq. (4)
    k.th = pth * iS;                                              // eq. (5)
    k.ph = fma((Sigma - 2.0 * r) * L, is2, -2.0 * a * r) * iS * iD;   // eq. (12)
    k.pr = iS * (fma(r, GiS, 2.0 * r * q) - (r - 1.0) * fma(q, q, pr2));
    k.pth = s * c * iS * (fma(L * L, is2 * is2, -a2) - a2 * GiS);
}

// ------------------------------------------------------------------------------------------------
// Embedded pairs (reading H).  TAB 0: Fehlberg 4(5) (BASELINE.json:configs[0] "RKF45");
// TAB 1: Cash–Karp (the pair of Press et al. 1992, cited PAPER.md:L90).
// ------------------------------------------------------------------------------------------------
template <int TAB>
__host__ __device__ constexpr double rk_a(int i, int j) {
    if (TAB == 0) {
        switch (i * 8 + j) {
            case 1 * 8 + 0: return 1.0 / 4.0;
            case 2 * 8 + 0: return 3.0 / 32.0;      case 2 * 8 + 1: return 9.0 / 32.0;
            case 3 * 8 + 0: return 1932.0 / 2197.0; case 3 * 8 + 1: return -7200.0 / 2197.0; case 3 * 8 + 2: return 7296.0 / 2197.0;
            case 4 * 8 + 0: return 439.0 / 216.0;   case 4 * 8 + 1: return -8.0;             case 4 * 8 + 2: return 3680.0 / 513.0;
            case 4 * 8 + 3: return -845.0 / 4104.0;
            case 5 * 8 + 0: return -8.0 / 27.0;     case 5 * 8 + 1: return 2.0;              case 5 * 8 + 2: return -3544.0 / 2565.0;
            case 5 * 8 + 3: return 1859.0 / 4104.0; case 5 * 8 + 4: return -11.0 / 40.0;
            default: return 0.0;
        }
    } else {
        switch (i * 8 + j) {
            case 1 * 8 + 0: return 1.0 / 5.0;
            case 2 * 8 + 0: return 3.0 / 40.0;      case 2 * 8 + 1: return 9.0 / 40.0;
            case 3 * 8 + 0: return 3.0 / 10.0;      case 3 * 8 + 1: return -9.0 / 10.0;      case 3 * 8 + 2: return 6.0 / 5.0;
            case 4 * 8 + 0: return -11.0 / 54.0;    case 4 * 8 + 1: return 5.0 / 2.0;        case 4 * 8 + 2: return -70.0 / 27.0;
            case 4 * 8 + 3: return 35.0 / 27.0;
            case 5 * 8 + 0: return 1631.0 / 55296.0; case 5 * 8 + 1: return 175.0 / 512.0;   case 5 * 8 + 2: return 575.0 / 13824.0;
            case 5 * 8 + 3: return 44275.0 / 110592.0; case 5 * 8 + 4: return 253.0 / 4096.0;
            default: return 0.0;
        }
    }
}

template <int TAB>
__host__ __device__ constexpr double rk_b5(int j) {
    if (TAB == 0) {
        switch (j) { case 0: return 16.0 / 135.0; case 2: return 6656.0 / 12825.0; case 3: return 28561.0 / 56430.0;
                     case 4: return -9.0 / 50.0;  case 5: return 2.0 / 55.0;       default: return 0.0; }
    } else {
        switch (j) { case 0: return 37.0 / 378.0; case 2: return 250.0 / 621.0; case 3: return 125.0 / 594.0;
                     case 5: return 512.0 / 1771.0; default: return 0.0; }
    }
}

template <int TAB>
__host__ __device__ constexpr double rk_b4(int j) {
    if (TAB == 0) {
        switch (j) { case 0: return 25.0 / 216.0; case 2: return 1408.0 / 2565.0; case 3: return 2197.0 / 4104.0;
                     case 4: return -1.0 / 5.0;   default: return 0.0; }
    } else {
        switch (j) { case 0: return 2825.0 / 27648.0; case 2: return 18575.0 / 48384.0; case 3: return 13525.0 / 55296.0;
                     case 4: return 277.0 / 14336.0;  case 5: return 1.0 / 4.0;         default: return 0.0; }
    }
}

// One attempt of size h from y with first slope k1: fifth-order result ynew and the error estimate
// yerr = h Σ (b5_j − b4_j) k_j (as Press et al.'s rkck forms it).  φ does not enter the right-hand
// side, so its stage values are never formed; only its two weighted sums are accumulated.
template <int TAB>
__device__ __forceinline__ void rk_attempt(const double a, const double a2, const double L,
                                           const State& y, const Slope& k1, const double h,
                                           State& ynew, State& yerr) {
    double kr[6], kt[6], kp[6], kq[6];      // slopes of r, θ, p_r, p_θ per stage (registers after unrolling)
    kr[0] = k1.r; kt[0] = k1.th; kp[0] = k1.pr; kq[0] = k1.pth;
    double ph5 = rk_b5<TAB>(0) * k1.ph;
    double phe = (rk_b5<TAB>(0) - rk_b4<TAB>(0)) * k1.ph;
#pragma unroll
    for (int i = 1; i < 6; ++i) {
        double sr = 0.0, st = 0.0, sp = 0.0, sq = 0.0;
#pragma unroll
        for (int j = 0; j < i; ++j) {
            const double aij = rk_a<TAB>(i, j);
            if (aij != 0.0) {
                sr = fma(aij, kr[j], sr); st = fma(aij, kt[j], st);
                sp = fma(aij, kp[j], sp); sq = fma(aij, kq[j], sq);
            }
        }
        Slope k; double s_, c_;
        geodesic_rhs(a, a2, L, fma(h, sr, y.r), fma(h, st, y.th), fma(h, sp, y.pr), fma(h, sq, y.pth), k, s_, c_);
        kr[i] = k.r; kt[i] = k.th; kp[i] = k.pr; kq[i] = k.pth;
        const double b5 = rk_b5<TAB>(i), be = rk_b5<TAB>(i) - rk_b4<TAB>(i);
        if (b5 != 0.0) ph5 = fma(b5, k.ph, ph5);
        if (be != 0.0) phe = fma(be, k.ph, phe);
    }
    double s5r = 0.0, s5t = 0.0, s5p = 0.0, s5q = 0.0, ser = 0.0, set = 0.0, sep = 0.0, seq = 0.0;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const double b5 = rk_b5<TAB>(j), be = rk_b5<TAB>(j) - rk_b4<TAB>(j);
        if (b5 != 0.0) { s5r = fma(b5, kr[j], s5r); s5t = fma(b5, kt[j], s5t); s5p = fma(b5, kp[j], s5p); s5q = fma(b5, kq[j], s5q); }
        if (be != 0.0) { ser = fma(be, kr[j], ser); set = fma(be, kt[j], set); sep = fma(be, kp[j], sep); seq = fma(be, kq[j], seq); }
    }
    ynew.r = fma(h, s5r, y.r); ynew.th = fma(h, s5t, y.th); ynew.ph = fma(h, ph5, y.ph);
    ynew.pr = fma(h, s5p, y.pr); ynew.pth = fma(h, s5q, y.pth);
    yerr.r = h * ser; yerr.th = h * set; yerr.ph = h * phe; yerr.pr = h * sep; yerr.pth = h * seq;
}

// Scaled max-norm of the error in units of rtol (reading G): scales (|r|, 1, 1, 1+|p_r|,
// 1+|p_θ|).  A NaN anywhere yields NaN (the attempt is then rejected with h × 0.1).
__device__ __forceinline__ double error_norm(const State& y, const State& e, const double rtol) {
    const double q0 = fabs(e.r) / fabs(y.r);
    const double q1 = fabs(e.th), q2 = fabs(e.ph);
    const double q3 = fabs(e.pr) / (1.0 + fabs(y.pr));
    const double q4 = fabs(e.pth) / (1.0 + fabs(y.pth));
    const double m = fmax(fmax(fmax(q0, q1), fmax(q2, q3)), q4);   // fmax drops NaNs …
    const double sum = q0 + q1 + q2 + q3 + q4;                     // … so detect them here (all q ≥ 0)
    return (sum != sum) ? sum : m / rtol;
}

// x^(-1/5) for x in (0, 1]: single-precision seed, two Newton steps y ← y (6 − x y⁵)/5 in FP64.
__device__ __forceinline__ double inv_fifth_root(const double x) {
    double y = (double)exp2f(-0.2f * log2f((float)x));
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const double y2 = y * y;
        const double y5 = y2 * y2 * y;
        y = y * fma(-x, y5, 6.0) * 0.2;
    }
    return y;
}

// ------------------------------------------------------------------------------------------------
// Camera: image-plane point (x, y) -> initial state, angular momentum L (E = −1).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void init_ray(const Params& P, const double x, const double yimg, State& y, double& L) {
    const double a = P.a, a2 = P.a2;
    // eqs. (18), (19) with z = 0
    const double Dd = P.R_obs * P.sin_obs - yimg * P.cos_obs;
    const double xp = Dd * P.cos_pobs - x * P.sin_pobs;
    const double yp = Dd * P.sin_pobs + x * P.cos_pobs;
    const double zp = P.r_obs * P.cos_obs + yimg * P.sin_obs;
    // eqs. (20)-(22)
    const double w = xp * xp + yp * yp + zp * zp - a2;
    const double r = sqrt(0.5 * (w + sqrt(w * w + 4.0 * a2 * zp * zp)));
    const double th = acos(zp / r);
    const double ph = atan2(yp, xp);
    // eqs. (24)-(26)
    const double R = sqrt(r * r + a2);
    double sP, cP, s, c;
    sincos(ph - P.phi_obs, &sP, &cP);
    sincos(th, &s, &c);
    const double Sigma = r * r + a2 * c * c;
    const double Delta = r * r - 2.0 * r + a2;
    const double rdot = -(r * R * s * P.sin_obs * cP + R * R * c * P.cos_obs) / Sigma;
    const double thdot = (r * s * P.cos_obs - R * c * P.sin_obs * cP) / Sigma;
    const double phdot = P.sin_obs * sP / (R * s);
    // eq. (7), μ = 0; E = −sqrt(E²) (reading B); eq. (8); eqs. (4), (5)
    const double E2 = ((Sigma - 2.0 * r) / (Sigma * Delta)) * (Sigma * rdot * rdot + Sigma * Delta * thdot * thdot)
                    + Delta * phdot * phdot * s * s;
    const double En = sqrt(E2);                                    // |E|
    const double Lraw = (Sigma * Delta * phdot + 2.0 * a * r * En) * s * s / (Sigma - 2.0 * r);
    const double inv = 1.0 / En;                                   // normalise to |E| = 1 (reading C)
    L = Lraw * inv;
    y.r = r; y.th = th; y.ph = ph;
    y.pr = Sigma * rdot / Delta * inv;
    y.pth = Sigma * thdot * inv;
}

}  // namespace ody
