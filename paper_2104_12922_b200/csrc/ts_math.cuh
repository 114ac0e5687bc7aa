// ts_math.cuh -- fp64 elementary functions for the control stage, sized for what the path needs
// (absolute error ~1e-16 on envelope values, relative ~2e-16 on increments) instead of libdevice's
// correctly-rounded-over-the-whole-range versions: ~35 instructions per pow instead of ~250, and no
// fp64 divisions.  Tables (768 B) are generated on the host in long double when the library starts
// and staged in shared memory by the kernel.
// Technique: the table-driven log2 (mantissa window [0.6875, 1.375) split into 2^-5 steps, table of reciprocals and
// logarithms of the interval centres, short polynomial in r = z/c - 1) and the exp2 with a `1.5 * 2^52` shift to split
// exponent, table index and remainder are the scheme used by open libm implementations (ARM optimized-routines /
// musl `log2`, `exp2`); table sizes, polynomial degrees and coefficients here are this code's own.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int TS_LOG_N = 32;  // sub-intervals of [0.6875, 1.375) for log2
constexpr int TS_EXP_N = 32;  // 2^(i/32)
constexpr unsigned long long TS_LOG_OFF = 0x3FE6000000000000ull;  // 0.6875

struct ts_math_tables {
    double invc[TS_LOG_N];  // ~1/c_i, c_i = centre of sub-interval i
    double logc[TS_LOG_N];  // -log2(invc[i]) rounded once
    double exp2t[TS_EXP_N]; // 2^(i/32)
};

#ifdef __CUDACC__
// Polynomial coefficients live in constant memory: an fp64 instruction takes a constant-bank operand directly, whereas a
// double literal in the code costs two extra moves per coefficient (the two 32-bit halves) in front of every DFMA.
struct ts_math_coefs {
    double log2p[10];   // log2(1+r) = r * sum_k log2p[k] r^k, log2p[k] = (-1)^k log2(e) / (k + 1)
    double exp2p[6];    // 2^f - 1 = f * sum_k exp2p[k] f^k, exp2p[k] = ln2^(k+1) / (k+1)!
    double expm1p[11];  // expm1(a) = a + a^2 * sum_k expm1p[k] a^k, expm1p[k] = 1 / (k+2)!
    double sin2pip[10]; // sin(pi y) = y * sum_k sin2pip[k] y^(2k)
};
__constant__ ts_math_coefs c_coef = {
    {1.4426950408889634, -1.4426950408889634 / 2.0, 1.4426950408889634 / 3.0, -1.4426950408889634 / 4.0, 1.4426950408889634 / 5.0,
     -1.4426950408889634 / 6.0, 1.4426950408889634 / 7.0, -1.4426950408889634 / 8.0, 1.4426950408889634 / 9.0, 0.0},
    {0.6931471805599453, 0.6931471805599453 * 0.6931471805599453 / 2.0, 0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 / 6.0,
     0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 / 24.0,
     0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 / 120.0,
     0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 * 0.6931471805599453 / 720.0},
    {0.5, 1.0 / 6.0, 1.0 / 24.0, 1.0 / 120.0, 1.0 / 720.0, 1.0 / 5040.0, 1.0 / 40320.0, 1.0 / 362880.0, 1.0 / 3628800.0,
     1.0 / 39916800.0, 1.0 / 479001600.0},
    {3.14159265358979312e+00, -5.16771278004997026e+00, 2.55016403987734552e+00, -5.99264529320792105e-01, 8.21458866111282326e-02,
     -7.37043094571435044e-03, 4.66302805767612554e-04, -2.19153534478302173e-05, 7.95205400147551261e-07, -2.29484289972698730e-08}};
// log2(x), x > 0 normal.  x = 2^k z, z in [0.6875, 1.375); r = z*invc - 1 (|r| < 0.0157, exact in an FMA up to
// 2^-59); log2 x = k + logc + log2(1+r).
__device__ __forceinline__ double ts_log2(double x, const ts_math_tables *T) {
    const unsigned long long ix = (unsigned long long)__double_as_longlong(x);
    const unsigned long long tmp = ix - TS_LOG_OFF;
    const int i = (int)(tmp >> (52 - 5)) & (TS_LOG_N - 1);
    const int k = (int)((long long)tmp >> 52);
    const double z = __longlong_as_double((long long)(ix - (tmp & 0xFFF0000000000000ull)));
    const double r = fma(z, T->invc[i], -1.0);
    // log2(1+r) = r * log2(e) * (1 - r/2 + r^2/3 - ...), degree 9 in r
    double p = c_coef.log2p[8];
#pragma unroll
    for (int k = 7; k >= 0; --k) p = fma(p, r, c_coef.log2p[k]);
    return fma(p, r, (double)k + T->logc[i]);
}

// 2^y for y in about [-1000, 1000] (callers clamp): y = n/32 + f, |f| <= 1/64.
__device__ __forceinline__ double ts_exp2(double y, const ts_math_tables *T) {
    const double big = 6755399441055744.0;  // 1.5 * 2^52
    const double kd = fma(y, 32.0, big);
    const int n = __double2loint(kd);        // rint(32 y)
    const double f = fma(kd - big, -1.0 / 32.0, y);
    // 2^f = exp(f ln2), degree 6
    double p = c_coef.exp2p[5];
#pragma unroll
    for (int k = 4; k >= 0; --k) p = fma(p, f, c_coef.exp2p[k]);
    const double t = T->exp2t[n & (TS_EXP_N - 1)];
    const double v = fma(t * p, f, t);
    const int e = n >> 5;
    return __hiloint2double(__double2hiint(v) + (e << 20), __double2loint(v));
}

// x^a for x in (0, 1], a > 0 (S4's ramp^alpha).  Absolute error ~1e-16.
__device__ __forceinline__ double ts_pow01(double x, double a, const ts_math_tables *T) {
    const double y = a * ts_log2(x, T);
    if (y < -1000.0) return 0.0;
    return ts_exp2(y, T);
}

// expm1(a) for |a| <= 0.125 by its series (relative accuracy down to a -> 0); libdevice beyond.
__device__ __forceinline__ double ts_expm1_small(double a) {
    if (fabs(a) > 0.125) return expm1(a);
    double p = c_coef.expm1p[10];          // 1/12!
#pragma unroll
    for (int k = 9; k >= 0; --k) p = fma(p, a, c_coef.expm1p[k]);
    return fma(p * a, a, a);
}
#endif
