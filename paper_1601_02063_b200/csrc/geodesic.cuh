// geodesic.cuh — device-side Kerr null-geodesic arithmetic of the Odyssey hot path.
//
//   init_ray      : pixel -> Boyer–Lindquist state and constants of motion, §2.2,
//                   eqs. (18)-(26), (7), (8), (4), (5).
//   geodesic_rhs  : the five right-hand sides, eqs. (4), (5), (12) and -dH/dr, -dH/dθ of the
//                   un-substituted Hamiltonian (≡ eqs. (14), (15) on the null shell; DESIGN.md
//                   reading A), pole clamp of PAPER.md:L90.
//   stage_point / rk_combine : stages 2..6 of an embedded 6-stage Runge–Kutta 5(4) pair ("fifth-
//                   order Runge–Kutta … adaptive step size", Press et al. 1992) with the first
//                   slope k1 supplied by the caller (it is cached across rejected attempts).
//
// Photon energy is normalised to E = -1 (ray traced backwards in time; readings B, C),
// which is folded into the formulas below: P = (r²+a²)E − aL = −Pm with Pm = r² + a² + aL.
#pragma once
#include "params.h"
#include "dmath.cuh"

namespace ody {

struct State { double r, th, ph, pr, pth; };     // y of PAPER.md:L88 without t
struct Slope { double r, th, ph, pr, pth, t; };  // dy/dλ; t (eq. (9)) is formed only by kernels that output time

// ------------------------------------------------------------------------------------------------
// Right-hand side.  Also returns sinθ, cosθ (unclamped) for the emission code.
// ------------------------------------------------------------------------------------------------
// The pole clamp of PAPER.md:L90 (reading I): |sinθ| < 1e-8 -> copysign(1e-8, sinθ).  The comparison is made on the
// bit patterns (for finite doubles |x| < |y| <=> bits(|x|) < bits(|y|) as integers): two integer compares and
// three selects on the ALU pipe instead of a DSETP, which would take an FP64-pipe slot in every right-hand side.
__device__ __forceinline__ double clamp_sin(const double s) {
    const int hi = __double2hiint(s), lo = __double2loint(s);
    const unsigned long long mag = ((unsigned long long)(unsigned)(hi & 0x7fffffff) << 32) | (unsigned)lo;
    const bool small = mag < 0x3E45798EE2308C3Aull;                // bits(1e-8)
    return small ? __hiloint2double((hi & 0x80000000) | 0x3E45798E, (int)0xE2308C3A) : s;
}

template <bool TIME = false>
__device__ __forceinline__ void geodesic_rhs(const double a, const double a2, const double L,
                                             const double r, const double th, const double pr, const double pth,
                                             Slope& k, double& sin_th, double& cos_th) {
    double s, c;
    d_sincos(th, s, c);
    sin_th = s; cos_th = c;
    s = clamp_sin(s);
    // 37 FP64 operations + three reciprocals (was 43): shared sub-expressions r² + a², 2q + G/Σ
    const double r2 = r * r;
    const double ra2 = r2 + a2;                                   // r² + a²
    const double Sigma = fma(a2, c * c, r2);                      // Σ = r² + a² cos²θ
    const double Delta = fma(-2.0, r, ra2);                       // Δ = r² − 2r + a²
    const double Pm = fma(a, L, ra2);                             // −P = r² + a² + aL  (E = −1)
    const double iS = d_rcp(Sigma), iD = d_rcp(Delta), is = d_rcp(s);   // three independent Newton chains
    const double is2 = is * is;
    const double D = fma(L, is, a * s);                           // L/sinθ − aE sinθ
    const double q = Pm * iD;                                     // −P/Δ
    const double pr2 = pr * pr;
    const double G = fma(Delta, pr2, fma(pth, pth, fma(D, D, -Pm * q)));   // 2ΣH
    const double GiS = G * iS;
    k.r = Delta * pr * iS;                                        // eq. (4)
    k.th = pth * iS;                                              // eq. (5)
    const double iSD = iS * iD;
    k.ph = fma(fma(-2.0, r, Sigma) * L, is2, -2.0 * a * r) * iSD;         // eq. (12)
    if (TIME) k.t = -fma(2.0 * r * Pm, iSD, 1.0);                         // eq. (9) with E = −1: −1 − 2r(r² + a² + aL)/(ΣΔ)
    k.pr = iS * fma(1.0 - r, fma(q, q, pr2), r * fma(2.0, q, GiS));
    k.pth = (s * c) * iS * fma(-a2, GiS, fma(L * L, is2 * is2, -a2));
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

// The same coefficients as __constant__ tables: the kernels read kRkA[TAB][i][j] etc. (compile-time
// indices; the constexpr functions above only prune the zero entries), so that the compiler loads them
// with LDCU.128 into uniform registers once, outside the stage loop, instead of building every
// 64-bit literal from two 32-bit immediates at each use.
#define ODY_ROW(T, i) { rk_a<T>(i, 0), rk_a<T>(i, 1), rk_a<T>(i, 2), rk_a<T>(i, 3), rk_a<T>(i, 4), 0.0 }
#define ODY_TABA(T) { ODY_ROW(T, 0), ODY_ROW(T, 1), ODY_ROW(T, 2), ODY_ROW(T, 3), ODY_ROW(T, 4), ODY_ROW(T, 5) }
#define ODY_B5(T) { rk_b5<T>(0), rk_b5<T>(1), rk_b5<T>(2), rk_b5<T>(3), rk_b5<T>(4), rk_b5<T>(5) }
#define ODY_BE(T) { rk_b5<T>(0) - rk_b4<T>(0), rk_b5<T>(1) - rk_b4<T>(1), rk_b5<T>(2) - rk_b4<T>(2), \
                    rk_b5<T>(3) - rk_b4<T>(3), rk_b5<T>(4) - rk_b4<T>(4), rk_b5<T>(5) - rk_b4<T>(5) }
__constant__ double kRkA[2][6][6] = { ODY_TABA(0), ODY_TABA(1) };
__constant__ double kRkB5[2][6] = { ODY_B5(0), ODY_B5(1) };
__constant__ double kRkBE[2][6] = { ODY_BE(0), ODY_BE(1) };
#undef ODY_ROW
#undef ODY_TABA
#undef ODY_B5
#undef ODY_BE

// The four dynamic components' slopes of the six stages (φ does not enter the right-hand side, so its
// stage values are never formed; only its two weighted sums are accumulated by the kernel).
// They live in shared memory, [component][stage][thread] — consecutive lanes hit consecutive 8-byte
// words, so every access is conflict-free.  This takes 48 registers off the kernel, which is what lets
// it run 5 blocks of 128 threads per SM at 96 registers without spills.
constexpr int STAGE_ROWS = 5;                           // r, θ, p_r, p_θ slopes + the absorption coefficient (RT scheme E')
constexpr int STAGE_SLOTS = 5;                          // k1..k5 are stored; the sixth slope goes from registers straight into the result
template <int NT>
struct StagesSmem {
    double* base;                                       // &smem[threadIdx.x]
    __device__ __forceinline__ double get(int c, int j) const { return base[(c * STAGE_SLOTS + j) * NT]; }
    __device__ __forceinline__ void set(int c, int j, double x) { base[(c * STAGE_SLOTS + j) * NT] = x; }
};

// Argument of stage I+1 (0-based I in 1..5): y + h Σ_{j<I} a_Ij k_j.
template <int TAB, int I, class KS>
__device__ __forceinline__ void stage_point(const KS& K, const State& y, const double h,
                                            double& r, double& th, double& pr, double& pth) {
    double sr = 0.0, st = 0.0, sp = 0.0, sq = 0.0;
#pragma unroll
    for (int j = 0; j < I; ++j) {
        if (rk_a<TAB>(I, j) != 0.0) {
            const double aij = kRkA[TAB][I][j];
            sr = fma(aij, K.get(0, j), sr); st = fma(aij, K.get(1, j), st);
            sp = fma(aij, K.get(2, j), sp); sq = fma(aij, K.get(3, j), sq);
        }
    }
    r = fma(h, sr, y.r); th = fma(h, st, y.th); pr = fma(h, sp, y.pr); pth = fma(h, sq, y.pth);
}

// Σ_{j<I} a_Ij v_j of row `c` (used for the stage values of τ in the Runge–Kutta-component transfer scheme).
template <int TAB, int I, class KS>
__device__ __forceinline__ double stage_sum(const KS& K, const int c) {
    double acc = 0.0;
#pragma unroll
    for (int j = 0; j < I; ++j)
        if (rk_a<TAB>(I, j) != 0.0) acc = fma(kRkA[TAB][I][j], K.get(c, j), acc);
    return acc;
}

// Fifth-order result and the error estimate h Σ (b5_j − b4_j) k_j (as Press et al.'s rkck forms it)
// of the four dynamic components; ph5 / phe are the kernel's running φ sums.
template <int TAB, class KS>
__device__ __forceinline__ void rk_combine(const KS& K, const Slope& k6, const State& y, const double h, const double ph5, const double phe,
                                           State& ynew, State& yerr) {
    double s5[4] = {0.0, 0.0, 0.0, 0.0}, se[4] = {0.0, 0.0, 0.0, 0.0};
    const double last[4] = {k6.r, k6.th, k6.pr, k6.pth};
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const bool has5 = rk_b5<TAB>(j) != 0.0, hase = (rk_b5<TAB>(j) - rk_b4<TAB>(j)) != 0.0;
        if (has5 || hase) {
            const double b5 = kRkB5[TAB][j], be = kRkBE[TAB][j];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const double k = (j < 5) ? K.get(c, j) : last[c];
                if (has5) s5[c] = fma(b5, k, s5[c]);
                if (hase) se[c] = fma(be, k, se[c]);
            }
        }
    }
    ynew.r = fma(h, s5[0], y.r); ynew.th = fma(h, s5[1], y.th); ynew.ph = fma(h, ph5, y.ph);
    ynew.pr = fma(h, s5[2], y.pr); ynew.pth = fma(h, s5[3], y.pth);
    yerr.r = h * se[0]; yerr.th = h * se[1]; yerr.ph = h * phe; yerr.pr = h * se[2]; yerr.pth = h * se[3];
}

// Scaled max-norm of the error in units of rtol (reading G): scales (|r|, 1, 1, 1+|p_r|,
// 1+|p_θ|).  The maximum is taken on the BIT PATTERNS of the five non-negative quotients: for non-negative doubles
// the integer order is the floating-point order, +inf sorts above every finite value and a NaN (0x7ff8…, sign
// cleared) above +inf, so a NaN anywhere comes out as NaN (the attempt is then rejected with h × 0.1) without a
// separate test — and the compares run on the ALU pipe, not on the FP64 pipe.  r > r_h > 0 on every live ray.
__device__ __forceinline__ long long abs_bits(const double x) { return __double_as_longlong(x) & 0x7fffffffffffffffLL; }
__device__ __forceinline__ double error_norm(const State& y, const State& e, const double inv_rtol) {
    const long long b0 = abs_bits(e.r * d_rcp(y.r));
    const long long b1 = abs_bits(e.th), b2 = abs_bits(e.ph);
    const long long b3 = abs_bits(e.pr * d_rcp(1.0 + fabs(y.pr)));
    const long long b4 = abs_bits(e.pth * d_rcp(1.0 + fabs(y.pth)));
    const long long m01 = b0 > b1 ? b0 : b1, m23 = b2 > b3 ? b2 : b3;
    const long long m = m01 > m23 ? m01 : m23;
    return __longlong_as_double(m > b4 ? m : b4) * inv_rtol;
}

// Step-size factor of the controller (reading G), one straight-line evaluation for both outcomes:
//   accepted attempt: min(5, 0.9 err^-1/5)  (5 below err = 1.889568e-4),   rejected: max(0.1, 0.9 err^-1/4).
// y = err^-1/n from a single-precision seed (MUFU.LG2 / MUFU.EX2, relative error d ~ 1e-6) and ONE third-order
// step y (1 + e/n + (n+1) e^2 / (2 n^2)), e = 1 - err y^n = -n d, which leaves (n+1)(2n+1)/(6 n^3) e^3 < 2e-17:
// the factor is correct to the rounding of its last operations.  Out-of-range arguments need no test: err = 0
// or denormal gives y = inf or NaN and the clamp returns 5; err = inf, NaN or > 1e38 gives 0 or NaN -> 0.1.
// (The first version branched: the two bodies ran one after the other in nearly every trip, the rejected one
// 6 lanes wide, and each was a serial chain of ~14 FP64 operations.)
__device__ __forceinline__ double step_factor(const double err, const bool accepted) {
    float l, sd;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"((float)err));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(sd) : "f"((accepted ? -0.2f : -0.25f) * l));
    const double y = (double)sd;
    const double y2 = y * y, y4 = y2 * y2;
    const double yn = accepted ? y4 * y : y4;
    const double e = fma(-err, yn, 1.0);
    const double p = fma(e, accepted ? 0.12 : 0.15625, accepted ? 0.2 : 0.25);
    const double f = 0.9 * fma(y * e, p, y);
    const double lim = accepted ? 5.0 : 0.1;
    return accepted ? (f < lim ? f : lim) : (f > lim ? f : lim);   // a NaN takes the limit in both cases
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
    const double r = d_sqrt(0.5 * (w + d_sqrt(w * w + 4.0 * a2 * zp * zp)));
    const double th = acos(zp * d_rcp(r));
    const double ph = atan2(yp, xp);
    // eqs. (24)-(26)
    const double R = d_sqrt(r * r + a2);
    double sP, cP, s, c;
    d_sincos(ph - P.phi_obs, sP, cP);
    d_sincos(th, s, c);
    const double Sigma = r * r + a2 * c * c;
    const double Delta = r * r - 2.0 * r + a2;
    const double iSig = d_rcp(Sigma), iDel = d_rcp(Delta), iS2r = d_rcp(Sigma - 2.0 * r);
    const double rdot = -(r * R * s * P.sin_obs * cP + R * R * c * P.cos_obs) * iSig;
    const double thdot = (r * s * P.cos_obs - R * c * P.sin_obs * cP) * iSig;
    const double phdot = P.sin_obs * sP * d_rcp(R * s);
    // eq. (7), μ = 0; E = −sqrt(E²) (reading B); eq. (8); eqs. (4), (5)
    const double E2 = ((Sigma - 2.0 * r) * iSig * iDel) * (Sigma * rdot * rdot + Sigma * Delta * thdot * thdot)
                    + Delta * phdot * phdot * s * s;
    const double inv = d_rsqrt(E2);                                // 1/|E|: normalise to |E| = 1 (reading C)
    const double En = E2 * inv;                                    // |E|
    const double Lraw = (Sigma * Delta * phdot + 2.0 * a * r * En) * s * s * iS2r;
    L = Lraw * inv;
    y.r = r; y.th = th; y.ph = ph;
    y.pr = Sigma * rdot * iDel * inv;
    y.pth = Sigma * thdot * inv;
}

}  // namespace ody
