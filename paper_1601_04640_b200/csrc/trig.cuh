// trig.cuh — branch-free sin/cos pair for the real-time nonlinear step (calcnu):
// psi <- psi exp(-i u), u = dt (V + G|psi|^2 + D Phi_dd).
//
// The CUDA library sincos carries a slow-path branch for huge arguments; sixteen calls in a row then
// run one after the other.  This version has no branch, so the compiler interleaves the sixteen
// evaluations of a thread (the fp64 pipe has an 8-cycle dependent latency on sm_100a).
//   k = nearest integer to u 2/pi;  r = u - k pi/2 with pi/2 as the sum of two doubles and FMAs
//   (pi/2 to 2^-106: the reduction error stays below 1e-23 for |k| < 2^30);  Taylor polynomials of sin r / cos r on |r| <= pi/4 up to
//   r^15 / r^16 (truncation < 5e-17);  quadrant from k mod 4.
// Absolute error <= 1.5e-16 against long-double sin/cos for |u| <= SINCOS_CW_MAX = 1e9 (checked on
// the host by tests/test_host_logic.py).  Beyond that — u = dt (V + G n + D Phi) of a meaningful time step is of
// order one — and for
// non-finite u, both results are NaN (a select, not a branch), as loud as the library's behaviour
// for infinities.
#pragma once
#include "cplx.cuh"

#define SINCOS_CW_MAX 1.0e9

// Coefficients: on the device they sit in constant memory, so that every DFMA takes its coefficient
// as a constant-bank operand (as 64-bit immediates they cost two uniform-register moves per use).
#define SINCOS_CW_COEFS                                                                                   \
    { 0.63661977236758134 /* 2/pi */, 1.5707963267948966, 6.123233995736766e-17, -1.4973849048591698e-33, \
      /* sin: -1/15!, 1/13!, -1/11!, 1/9!, -1/7!, 1/5!, -1/3! */                                          \
      -1.0 / 1307674368000.0, 1.0 / 6227020800.0, -1.0 / 39916800.0, 1.0 / 362880.0, -1.0 / 5040.0,       \
      1.0 / 120.0, -1.0 / 6.0,                                                                            \
      /* cos: 1/16!, -1/14!, 1/12!, -1/10!, 1/8!, -1/6!, 1/4!, -1/2! */                                   \
      1.0 / 20922789888000.0, -1.0 / 87178291200.0, 1.0 / 479001600.0, -1.0 / 3628800.0, 1.0 / 40320.0,   \
      -1.0 / 720.0, 1.0 / 24.0, -0.5 }
#if defined(__CUDACC__)
static __constant__ double sincos_cw_dev[19] = SINCOS_CW_COEFS;
#endif
static const double sincos_cw_host[19] = SINCOS_CW_COEFS;

DBEC_HD void sincos_cw(double u, double* sn, double* cs) {
#if defined(__CUDA_ARCH__)
    const double* K = sincos_cw_dev;
#else
    const double* K = sincos_cw_host;
#endif
    // out of range or not finite -> NaN, by a select of a constant (a division here would put a branch with a
    // slow-path call around every evaluation and keep the compiler from interleaving them)
#if defined(__CUDA_ARCH__)
    u = (fabs(u) <= SINCOS_CW_MAX) ? u : __longlong_as_double(0x7ff8000000000000LL);
#else
    { union { unsigned long long i; double d; } qn; qn.i = 0x7ff8000000000000ULL; u = (fabs(u) <= SINCOS_CW_MAX) ? u : qn.d; }
#endif
    const double MAGIC = 6755399441055744.0;                 // 1.5 * 2^52: adding it rounds to nearest integer
    const double kb = fma(u, K[0], MAGIC);
    const double kd = kb - MAGIC;
#if defined(__CUDA_ARCH__)
    const int q = __double2loint(kb);
#else
    union { double d; unsigned long long u; } cv; cv.d = kb;
    const int q = (int)(unsigned)(cv.u & 0xffffffffull);
#endif
    double r = fma(-kd, K[1], u);
    r = fma(-kd, K[2], r);
    const double r2 = r * r;
    double ps = K[4];
#pragma unroll
    for (int i = 5; i <= 10; ++i) ps = fma(ps, r2, K[i]);
    const double sr = fma(ps * r2, r, r);
    double pc = K[11];
#pragma unroll
    for (int i = 12; i <= 18; ++i) pc = fma(pc, r2, K[i]);
    const double cr = fma(pc, r2, 1.0);
    const double a = (q & 1) ? cr : sr;                      // sin u up to sign
    const double b = (q & 1) ? sr : cr;                      // cos u up to sign
    *sn = (q & 2) ? -a : a;
    *cs = ((q + 1) & 2) ? -b : b;
}

// ---- branch-free exp for the imaginary-time nonlinear step: psi <- psi exp(-u) ----
// The library exp has a slow-path branch (results near the subnormal range), which keeps the compiler from
// interleaving the evaluations of a thread just as the library sincos does.  Here:
//   k = nearest integer to x log2(e);  r = x - k ln2 with ln2 as the sum of two doubles (|r| <= 0.3466);
//   Taylor polynomial of exp r up to r^13 (truncation < 5e-18 relative);  result = p 2^k, the scaling done as two
//   multiplications by 2^(k/2) so that overflow gives inf and underflow goes through the subnormals to 0.
// Relative error <= 2.5e-16 against long-double exp on |x| <= 700 (tests/test_host_logic.py); x is clamped to
// [-750, 750] first (exp(-750) = 0, exp(750) = inf in fp64 anyway); NaN in, NaN out (a select).
#define EXP_CW_COEFS                                                                                         \
    { 1.4426950408889634 /* log2 e */, 0.6931471805599453 /* ln2 hi */, 2.3190468138462996e-17 /* ln2 lo */, \
      1.0 / 6227020800.0, 1.0 / 479001600.0, 1.0 / 39916800.0, 1.0 / 3628800.0, 1.0 / 362880.0,              \
      1.0 / 40320.0, 1.0 / 5040.0, 1.0 / 720.0, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0, 0.5 }
#if defined(__CUDACC__)
static __constant__ double exp_cw_dev[15] = EXP_CW_COEFS;
#endif
static const double exp_cw_host[15] = EXP_CW_COEFS;

DBEC_HD double exp_cw(double x) {
#if defined(__CUDA_ARCH__)
    const double* K = exp_cw_dev;
#else
    const double* K = exp_cw_host;
#endif
    const double xc = fmin(fmax(x, -750.0), 750.0);           // (NaN becomes -750 here; restored by the select below)
    const double MAGIC = 6755399441055744.0;                 // 1.5 * 2^52
    const double kb = fma(xc, K[0], MAGIC);
    const double kd = kb - MAGIC;
    double r = fma(-kd, K[1], xc);
    r = fma(-kd, K[2], r);
    double p = K[3];
#pragma unroll
    for (int i = 4; i <= 14; ++i) p = fma(p, r, K[i]);       // 1/13! r^11 + ... + 1/2
    p = fma(p * r, r, r) + 1.0;                              // 1 + r + r^2 (...)
#if defined(__CUDA_ARCH__)
    const int k = __double2loint(kb);
    const int k1 = k >> 1, k2 = k - k1;
    const double s1 = __hiloint2double((k1 + 1023) << 20, 0), s2 = __hiloint2double((k2 + 1023) << 20, 0);
#else
    union { double d; unsigned long long u; } cv; cv.d = kb;
    const int k = (int)(unsigned)(cv.u & 0xffffffffull);
    const int k1 = k >> 1, k2 = k - k1;
    union { unsigned long long u; double d; } a, b;
    a.u = (unsigned long long)(k1 + 1023) << 52; b.u = (unsigned long long)(k2 + 1023) << 52;
    const double s1 = a.d, s2 = b.d;
#endif
    const double e = (p * s1) * s2;
    return (x != x) ? x : e;
}
