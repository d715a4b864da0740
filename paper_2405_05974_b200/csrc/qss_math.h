// Internal: branch-free fp64 exp for the rate-constant phase (two exp per reaction dominate the wdot work,
// DESIGN.md "Roofline").  libdevice's exp spends ~3/4 of its instructions outside the fp64 pipe (special-case paths);
// rate-constant arguments are finite, so this version has no branches:
//   n = rint(x log2 e) by the 1.5*2^52 trick, r = x - n ln2 (Cody-Waite, two constants), exp(r) by a degree-13 Taylor
//   polynomial in Horner form (|r| <= 0.3466, truncation 4e-18), scaling by 2^n as two exponent-field factors so that
//   results down to the denormals and up to overflow round correctly.  Measured against float128 expq on 10^7 arguments
//   in [-745, 709]: max error 1.0 ulp, 0.86 ulp outside the denormal range (tests/test_host_logic.py compiles this
//   header for the host and repeats the measurement with a 1.5 ulp bound).
// Preconditions: |x| < 2^30 (NaN gives NaN; +-inf gives NaN, not inf / 0); arguments that may be larger (fall-off
// placeholders) go through qss_exp_sat below.
#ifndef QSS_MATH_H
#define QSS_MATH_H
#include "qss_stdint.h"
#ifndef __CUDACC_RTC__
#include <string.h>
#endif

#ifdef __CUDACC__
#define QSS_HD __host__ __device__ __forceinline__
#else
#define QSS_HD inline
#include <cmath>
#endif

QSS_HD double qss_pow2_factor(int e) {      // 2^e for -1022 <= e <= 1023
#ifdef __CUDA_ARCH__
    return __hiloint2double((e + 1023) << 20, 0);
#else
    const uint64_t b = (uint64_t)(e + 1023) << 52;
    double d;
    memcpy(&d, &b, 8);
    return d;
#endif
}

QSS_HD double qss_exp(double x) {
    const double kShift = 6755399441055744.0;                 // 1.5 * 2^52
    const double kL2E = 1.4426950408889634074;
    const double kLn2Hi = 6.93147180369123816490e-01;          // ln 2, high part (low 21 mantissa bits zero)
    const double kLn2Lo = 1.90821492927058770002e-10;
    const double t = fma(x, kL2E, kShift);
#ifdef __CUDA_ARCH__
    int n = __double2loint(t);
#else
    uint64_t tb;
    memcpy(&tb, &t, 8);
    int n = (int)(uint32_t)tb;
#endif
    const double nf = t - kShift;
    double r = fma(nf, -kLn2Hi, x);
    r = fma(nf, -kLn2Lo, r);
    double q = 1.6059043836821613e-10;                         // 1/13!
    q = fma(q, r, 2.08767569878681e-09);                       // 1/12!
    q = fma(q, r, 2.505210838544172e-08);                      // 1/11!
    q = fma(q, r, 2.755731922398589e-07);                      // 1/10!
    q = fma(q, r, 2.7557319223985893e-06);                     // 1/9!
    q = fma(q, r, 2.48015873015873e-05);                       // 1/8!
    q = fma(q, r, 1.984126984126984e-04);                      // 1/7!
    q = fma(q, r, 1.388888888888889e-03);                      // 1/6!
    q = fma(q, r, 8.333333333333333e-03);                      // 1/5!
    q = fma(q, r, 4.1666666666666664e-02);                     // 1/4!
    q = fma(q, r, 1.6666666666666666e-01);                     // 1/3!
    q = fma(q, r, 0.5);
    q = fma(q, r, 1.0);
    q = fma(q, r, 1.0);
    n = n < -2000 ? -2000 : (n > 2000 ? 2000 : n);             // keeps both exponent fields valid for any finite x
    const int n1 = n >> 1, n2 = n - n1;
    return q * qss_pow2_factor(n1) * qss_pow2_factor(n2);
}

// exp for arguments that may lie far outside [-745, 709] (CHEMKIN placeholder Troe temperatures: -T/1e-30, -1e30/T):
// saturates to exp(-746) = 0 and exp(710) = inf like the library function (NaN stays NaN).
QSS_HD double qss_exp_sat(double x) {
    return qss_exp(x < -746.0 ? -746.0 : (x > 710.0 ? 710.0 : x));
}

// The same exponential with the polynomial in Estrin form: 13 FMA + 3 multiplications in a dependent chain of depth 4
// instead of 13 (the rate phase of kernel variant 3 is bound by the latency of these chains, not by the fp64 pipe).
// Same argument reduction and scaling; the extra roundings at magnitude ~1 cost < 1 ulp (max error 2 ulp).
QSS_HD double qss_exp_e(double x) {
    const double kShift = 6755399441055744.0;                 // 1.5 * 2^52
    const double kL2E = 1.4426950408889634074;
    const double kLn2Hi = 6.93147180369123816490e-01;
    const double kLn2Lo = 1.90821492927058770002e-10;
    const double t = fma(x, kL2E, kShift);
#ifdef __CUDA_ARCH__
    int n = __double2loint(t);
#else
    uint64_t tb;
    memcpy(&tb, &t, 8);
    int n = (int)(uint32_t)tb;
#endif
    const double nf = t - kShift;
    double r = fma(nf, -kLn2Hi, x);
    r = fma(nf, -kLn2Lo, r);
    const double r2 = r * r, r4 = r2 * r2, r8 = r4 * r4;
    const double a0 = fma(r, 1.0, 1.0), a1 = fma(r, 1.6666666666666666e-01, 0.5);
    const double a2 = fma(r, 8.333333333333333e-03, 4.1666666666666664e-02), a3 = fma(r, 1.984126984126984e-04, 1.388888888888889e-03);
    const double a4 = fma(r, 2.7557319223985893e-06, 2.48015873015873e-05), a5 = fma(r, 2.505210838544172e-08, 2.755731922398589e-07);
    const double a6 = fma(r, 1.6059043836821613e-10, 2.08767569878681e-09);
    const double b0 = fma(a1, r2, a0), b1 = fma(a3, r2, a2), b2 = fma(a5, r2, a4);
    const double d0 = fma(b1, r4, b0), d1 = fma(a6, r4, b2);
    const double q = fma(d1, r8, d0);
    n = n < -2000 ? -2000 : (n > 2000 ? 2000 : n);
    const int n1 = n >> 1, n2 = n - n1;
    return q * qss_pow2_factor(n1) * qss_pow2_factor(n2);
}

// Reciprocal of a positive normal double without the special-case paths of the IEEE division (the generic 1/x costs
// ~80 instructions, x/y ~136, and the fall-off path has six of them): hardware seed (20+ bits) + two Newton steps in
// FMA form, result within ~1 ulp.  Host builds use the plain division.
QSS_HD double qss_rcp(double x) {
#ifdef __CUDA_ARCH__
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    return r;
#else
    return 1.0 / x;
#endif
}

// The same function with a table of 2^(j/64), j = 0..63: exp(x) = 2^k 2^(j/64) exp(r), |r| <= ln2/128, exp(r) by a polynomial of
// degree 5 (truncation 3.5e-17): 12 fp64 operations instead of 22.  `tab` is whatever QSS_EXP_TAB_LOAD reads element j from (a
// pointer by default; the kernels define the macro as a shared-memory read).  Valid for |x| < 2^24 like qss_exp; max error 1 ulp.
#ifndef QSS_EXP_TAB_LOAD
#define QSS_EXP_TAB_LOAD(tab, j) ((tab)[j])
#endif
template <class TAB>
QSS_HD double qss_exp_tab(double x, TAB tab) {
    const double kShift = 6755399441055744.0;                 // 1.5 * 2^52
    const double k64L2E = 92.33248261689366;                  // 64 / ln 2
    const double kHi = 0.01083042469326756;                   // ln 2 / 64, 32 significant bits (n kHi is exact for |n| < 2^20)
    const double kLo = 2.9815858269852933e-12;
    const double t = fma(x, k64L2E, kShift);
#ifdef __CUDA_ARCH__
    int n = __double2loint(t);
#else
    uint64_t tb;
    memcpy(&tb, &t, 8);
    int n = (int)(uint32_t)tb;
#endif
    const double nf = t - kShift;
    double r = fma(nf, -kHi, x);
    r = fma(nf, -kLo, r);
    const double r2 = r * r;
    const double a1 = fma(r, 1.6666666666666666e-01, 0.5), a2 = fma(r, 8.333333333333333e-03, 4.1666666666666664e-02);
    const double p = fma(fma(a2, r2, a1), r2, r);              // exp(r) - 1
    n = n < -128000 ? -128000 : (n > 128000 ? 128000 : n);     // keeps both exponent fields valid for any finite x
    const double tj = QSS_EXP_TAB_LOAD(tab, n & 63);
    const int k = n >> 6, k1 = k >> 1, k2 = k - k1;
    return fma(tj, p, tj) * qss_pow2_factor(k1) * qss_pow2_factor(k2);
}

#endif
