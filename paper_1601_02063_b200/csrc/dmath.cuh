// dmath.cuh — branch-free FP64 elementary functions for the Odyssey kernels.
//
// The CUDA math library's double-precision 1/x, sqrt, sincos, exp, log, expm1 each carry a slow path
// (denormals, huge arguments) behind a branch.  In the fused geodesic + radiative-transfer loop those
// branches (a) split the code into small basic blocks, so the scheduler cannot interleave the
// independent dependency chains of one right-hand-side evaluation, and (b) add code that has to live
// in the instruction cache.  The arguments on the hot path are all of ordinary magnitude (radii,
// angles of a few radians, optical depths, exponents clamped to +-700), so the versions below do the
// fast path only, straight-line:
//
//   d_rcp, d_rsqrt, d_sqrt : hardware seed (MUFU.RCP64H / MUFU.RSQ64H) + Newton steps in FMA
//   d_sincos               : two-term Cody–Waite reduction by pi/2, odd/even polynomials on [-pi/4, pi/4]
//   d_exp, d_expm1         : x = k ln2 + r, e^r = 1 + r q(r), scaling through the exponent field
//   d_log                  : x = 2^e m, m in [sqrt(1/2), sqrt(2)), log m = 2 atanh((m-1)/(m+1))
//
// Accuracy: a few ulp (tests/test_dmath.py: the host build of this header against libm, and the device build
// through odyssey_eval_math against libm and scipy).  Polynomial tables: dmath_coeffs.h (gen_dmath_coeffs.py).
#pragma once
#include <stdint.h>
#include "dmath_coeffs.h"

// Under nvcc the functions are device-only and every polynomial table is a __constant__ array: the
// compiler then fetches coefficients two at a time with LDCU.128 into uniform registers and hoists the
// loads out of the stage loop, instead of materialising each 64-bit literal with two UMOV/IMAD.MOV
// instructions at every use (20 % of all issued instructions in the first version of the kernel).
// Under a host compiler (tests/dmath_host.cpp) the same tables are plain static arrays.
#if defined(__CUDACC__)
#define ODY_HD __device__ __forceinline__
#define ODY_TABLE __constant__ double
#define ODY_TABLE_F __constant__ float
#else
#define ODY_HD inline
#define ODY_TABLE static const double
#define ODY_TABLE_F static const float
#endif

namespace ody {

#define ODY_COEF(i, v) v,
ODY_TABLE kSinS[ODY_SINS_N] = { ODY_SINS(ODY_COEF) };
ODY_TABLE kCosC[ODY_COSC_N] = { ODY_COSC(ODY_COEF) };
ODY_TABLE kExpQ[ODY_EXPQ_N] = { ODY_EXPQ(ODY_COEF) };
ODY_TABLE kLogP[ODY_LOGP_N] = { ODY_LOGP(ODY_COEF) };
#define ODY_COEFF(i, v) (float)(v),
ODY_TABLE_F kExpQf[ODY_EXPQF_N] = { ODY_EXPQF(ODY_COEFF) };
ODY_TABLE_F kLogPf[ODY_LOGPF_N] = { ODY_LOGPF(ODY_COEFF) };
#undef ODY_COEFF
// scalar constants that do not fit a 32-bit immediate (low word non-zero)
ODY_TABLE kDm[10] = {
    6755399441055744.0,             // 0: 1.5 * 2^52, round-to-nearest-integer trick
    0.63661977236758134308,         // 1: 2/pi
    1.57079632679489655800e+00,     // 2: pi/2 high part
    6.12323399573676603587e-17,     // 3: pi/2 low part
    1.44269504088896338700e+00,     // 4: 1/ln2
    6.93147180559945286227e-01,     // 5: ln2 (nearest double)
    2.31904681384629955842e-17,     // 6: ln2 - (5)
    6.93147180369123816490e-01,     // 7: ln2 high part (32 bits: e * this is exact)
    1.90821492927058770002e-10,     // 8: ln2 - (7)
    0.0 };
#undef ODY_COEF

ODY_HD double d_from_bits(uint64_t u) {
#if defined(__CUDA_ARCH__)
    return __longlong_as_double((long long)u);
#else
    double d; __builtin_memcpy(&d, &u, 8); return d;
#endif
}
ODY_HD uint64_t d_to_bits(double d) {
#if defined(__CUDA_ARCH__)
    return (uint64_t)__double_as_longlong(d);
#else
    uint64_t u; __builtin_memcpy(&u, &d, 8); return u;
#endif
}
ODY_HD int32_t d_lo_word(double d) {
#if defined(__CUDA_ARCH__)
    return __double2loint(d);
#else
    return (int32_t)(uint32_t)d_to_bits(d);
#endif
}
// x with its sign flipped when bit 31 of `mask_hi` is set (one LOP3 on the high word)
ODY_HD double d_xor_sign(double x, uint32_t mask_hi) {
#if defined(__CUDA_ARCH__)
    return __hiloint2double(__double2hiint(x) ^ (int)(mask_hi & 0x80000000u), __double2loint(x));
#else
    return d_from_bits(d_to_bits(x) ^ ((uint64_t)(mask_hi & 0x80000000u) << 32));
#endif
}
// 2^k for -1022 <= k <= 1023
ODY_HD double d_pow2i(int32_t k) {
#if defined(__CUDA_ARCH__)
    return __hiloint2double((k + 1023) << 20, 0);
#else
    return d_from_bits((uint64_t)(uint32_t)(k + 1023) << 52);
#endif
}
ODY_HD double d_fma(double a, double b, double c) {
#if defined(__CUDA_ARCH__)
    return fma(a, b, c);
#else
    return __builtin_fma(a, b, c);
#endif
}

// ---- hardware seeds: MUFU.RCP64H / RSQ64H fill the high word only, i.e. 20 mantissa bits (measured on
// B200: max relative error 2^-19.96 and 2^-20.08); the host versions (same truncation) exist for the CPU test
ODY_HD double d_rcp_seed(double x) {
#if defined(__CUDA_ARCH__)
    double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y;
#else
    return d_from_bits(d_to_bits(1.0 / x) & 0xffffffff00000000ull);
#endif
}
ODY_HD double d_rsqrt_seed(double x) {
#if defined(__CUDA_ARCH__)
    double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y;
#else
    return d_from_bits(d_to_bits(1.0 / __builtin_sqrt(x)) & 0xffffffff00000000ull);
#endif
}

// 1/x for normal x (no zero, infinity, NaN or denormal handling).  One third-order step from the 20-bit
// seed: y (1 + e + e^2), e = 1 - x y, leaves a relative error e^3 = 2^-60.
ODY_HD double d_rcp(double x) {
    const double y = d_rcp_seed(x);
    double e = d_fma(-x, y, 1.0);
    e = d_fma(e, e, e);                 // e + e^2
    return d_fma(y, e, y);
}

// x^-1/2 for normal x > 0.  One third-order step: y (1 + e/2 + 3 e^2/8), e = 1 - x y^2 (error ~ e^3 5/16).
ODY_HD double d_rsqrt(double x) {
    const double y = d_rsqrt_seed(x);
    const double e = d_fma(-x, y * y, 1.0);
    return d_fma(y * e, d_fma(e, 0.375, 0.5), y);
}

// sqrt(x) for normal x > 0 (x = 0 gives NaN: callers guard).
ODY_HD double d_sqrt(double x) {
    const double y = d_rsqrt(x);
    const double s = x * y;
    return d_fma(d_fma(-s, s, x), 0.5 * y, s);
}

// sin and cos of an angle of ordinary size (|x| < ~1e5; accuracy degrades slowly beyond).
ODY_HD void d_sincos(double x, double& sn, double& cs) {
    const double* const S = kSinS; const double* const C = kCosC;
    const double MAGIC = kDm[0];
    const double t = d_fma(x, kDm[1], MAGIC);                      // x * 2/pi
    const int32_t q = d_lo_word(t);                                // low word = nearest integer
    const double k = t - MAGIC;
    double r = d_fma(-k, kDm[2], x);                               // pi/2 high part
    r = d_fma(-k, kDm[3], r);                                      // pi/2 low part
    const double z = r * r;
    double ps = S[ODY_SINS_N - 1], pc = C[ODY_COSC_N - 1];
#if defined(__CUDA_ARCH__)
#pragma unroll
#endif
    for (int i = ODY_SINS_N - 2; i >= 0; --i) { ps = d_fma(ps, z, S[i]); pc = d_fma(pc, z, C[i]); }
    const double sr = d_fma(ps * z, r, r);                         // r + r^3 S(z)
    const double cr = d_fma(z, d_fma(z, pc, -0.5), 1.0);           // 1 - z/2 + z^2 C(z), Horner: both constants are 32-bit immediates
    const bool swap = q & 1;
    const double s0 = swap ? cr : sr, c0 = swap ? sr : cr;
    sn = d_xor_sign(s0, (uint32_t)q << 30);                        // negative in quadrants 2, 3
    cs = d_xor_sign(c0, (uint32_t)(q + 1) << 30);                  // negative in quadrants 1, 2
}

// x = k ln2 + r with |r| <= ln2/2; returns r and 2^k (as a double), for |x| <= ~700.
ODY_HD double d_exp_reduce(double x, double& two_k) {
    const double MAGIC = kDm[0];
    const double t = d_fma(x, kDm[4], MAGIC);
    const int32_t k = d_lo_word(t);
    const double kf = t - MAGIC;
    double r = d_fma(-kf, kDm[5], x);
    r = d_fma(-kf, kDm[6], r);
    two_k = d_pow2i(k);
    return r;
}

ODY_HD double d_expq(double r) {                                   // (e^r - 1)/r
    const double* const Q = kExpQ;
    double p = Q[ODY_EXPQ_N - 1];
#if defined(__CUDA_ARCH__)
#pragma unroll
#endif
    for (int i = ODY_EXPQ_N - 2; i >= 0; --i) p = d_fma(p, r, Q[i]);
    return p;
}

// e^x for |x| <= 700 (no range check: the caller knows the range).
ODY_HD double d_exp_nc(double x) {
    double two_k;
    const double r = d_exp_reduce(x, two_k);
    return d_fma(r * d_expq(r), two_k, two_k);                     // 2^k (1 + r q)
}

// e^x for x <= 700; arguments below -700 (and NaN) return 0.
ODY_HD double d_exp_lo(double x) {
    const bool ok = x >= -700.0;
    const double v = d_exp_nc(ok ? x : -700.0);
    return ok ? v : 0.0;
}

// e^x; arguments below -700 return 0, above 700 are clamped.
ODY_HD double d_exp(double x) { return d_exp_lo(x > 700.0 ? 700.0 : x); }

// e^x - 1, accurate near 0, for |x| <= 700.
ODY_HD double d_expm1_nc(double x) {
    double two_k;
    const double r = d_exp_reduce(x, two_k);
    return d_fma(r * d_expq(r), two_k, two_k - 1.0);               // 2^k r q + (2^k - 1)
}

// e^x - 1 with the argument clamped to [-700, 700] (e^-700 - 1 = -1 exactly in FP64).
ODY_HD double d_expm1(double x) { return d_expm1_nc(x < -700.0 ? -700.0 : (x > 700.0 ? 700.0 : x)); }

// ---- mixed-precision variants: argument reduction and reconstruction in FP64 — the integer
// part of an exponent must not lose bits — and only the polynomial core on the reduced argument in FP32
// (relative error ~1e-7).  Used by the PREC = 1 transfer code only.
ODY_HD float f_fmaf(float a, float b, float c) {
#if defined(__CUDA_ARCH__)
    return fmaf(a, b, c);
#else
    return __builtin_fmaf(a, b, c);
#endif
}
ODY_HD float f_expq(float r) {
    float p = kExpQf[ODY_EXPQF_N - 1];
#if defined(__CUDA_ARCH__)
#pragma unroll
#endif
    for (int i = ODY_EXPQF_N - 2; i >= 0; --i) p = f_fmaf(p, r, kExpQf[i]);
    return p;
}
ODY_HD double f_exp_nc(double x) {
    double two_k;
    const float r = (float)d_exp_reduce(x, two_k);
    return d_fma((double)(r * f_expq(r)), two_k, two_k);
}
ODY_HD double f_exp(double x) {
    const bool ok = x >= -700.0;
    const double v = f_exp_nc(ok ? (x > 700.0 ? 700.0 : x) : -700.0);
    return ok ? v : 0.0;
}
ODY_HD double f_expm1_nc(double x) {
    double two_k;
    const float r = (float)d_exp_reduce(x, two_k);
    return d_fma((double)(r * f_expq(r)), two_k, two_k - 1.0);
}
ODY_HD double f_log(double x) {
    const uint64_t u = d_to_bits(x);
    const uint64_t adj = u + 0x00095f619980c433ull;
    const int32_t e = (int32_t)(adj >> 52) - 1023;
    const float f = (float)(d_from_bits(u - ((uint64_t)(int64_t)e << 52)) - 1.0);
#if defined(__CUDA_ARCH__)
    const float s = __fdividef(f, 2.0f + f);
#else
    const float s = f / (2.0f + f);
#endif
    const float z = s * s;
    float p = kLogPf[ODY_LOGPF_N - 1];
#if defined(__CUDA_ARCH__)
#pragma unroll
#endif
    for (int i = ODY_LOGPF_N - 2; i >= 0; --i) p = f_fmaf(p, z, kLogPf[i]);
    const double ef = (double)e;
    return d_fma(ef, kDm[7], (double)(2.0f * s * p) + ef * kDm[8]);
}

// natural logarithm of a normal x > 0.
ODY_HD double d_log(double x) {
    const double* const P = kLogP;
    const uint64_t u = d_to_bits(x);
    // exponent chosen so that the mantissa m lies in [sqrt(1/2), sqrt(2)): add (1 - sqrt(1/2)) in the mantissa field
    const uint64_t adj = u + 0x00095f619980c433ull;                // bits(1.0) - bits(sqrt(1/2))
    const int32_t e = (int32_t)(adj >> 52) - 1023;
    const double m = d_from_bits(u - ((uint64_t)(int64_t)e << 52));
    const double f = m - 1.0;
    const double s = f * d_rcp(2.0 + f);
    const double z = s * s;
    double p = P[ODY_LOGP_N - 1];
#if defined(__CUDA_ARCH__)
#pragma unroll
#endif
    for (int i = ODY_LOGP_N - 2; i >= 0; --i) p = d_fma(p, z, P[i]);
    const double ef = (double)e;
    // log x = e ln2 + 2 s p(z), ln2 split so that e * ln2_hi is exact
    return d_fma(ef, kDm[7], d_fma(2.0 * s, p, ef * kDm[8]));
}

}  // namespace ody
