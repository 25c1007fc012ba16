// trig.cuh — branch-free sin/cos pair for the real-time nonlinear step (calcnu):
// psi <- psi exp(-i u), u = dt (V + G|psi|^2 + D Phi_dd).
//
// The CUDA library sincos carries a slow-path branch for huge arguments; sixteen calls in a row then
// run one after the other.  This version has no branch, so the compiler interleaves the sixteen
// evaluations of a thread (the fp64 pipe has an 8-cycle dependent latency on sm_100a).
//   k = nearest integer to u 2/pi;  r = u - k pi/2 with pi/2 as the sum of two doubles and FMAs
//   (pi/2 to 2^-106: the reduction error stays below 1e-23 for |k| < 2^30);  minimax polynomials of sin r / cos r on
//   |r| <= pi/4 up to r^13 / r^14 (trig_coefficients.py, a Remez fit in 60-digit arithmetic: 4e-18 / 2e-19 absolute);  quadrant from k mod 4.
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
    { 0.63661977236758134 /* 2/pi */, 1.5707963267948966, 6.123233995736766e-17,                          \
      /* sin r = r + r^3 P(r^2), coefficients of r^13 ... r^3 */                                          \
      1.5894743283863398e-10, -2.505073511868829e-08, 2.7557313655187267e-06,                       \
      -0.00019841269830153272, 0.008333333333323673, -0.16666666666666644,                          \
      /* cos r = 1 - r^2/2 + r^4 Q(r^2), coefficients of r^14 ... r^4 */                                  \
      -1.1368002341468553e-11, 2.0875898081312824e-09, -2.7557315740699307e-07,                      \
      2.480158729463356e-05, -0.0013888888888882846, 0.04166666666666665, -0.5 }
#if defined(__CUDACC__)
static __constant__ double sincos_cw_dev[16] = SINCOS_CW_COEFS;
#endif
static const double sincos_cw_host[16] = SINCOS_CW_COEFS;

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
    double ps = K[3];
#pragma unroll
    for (int i = 4; i <= 8; ++i) ps = fma(ps, r2, K[i]);
    const double sr = fma(ps * r2, r, r);
    double pc = K[9];
#pragma unroll
    for (int i = 10; i <= 15; ++i) pc = fma(pc, r2, K[i]);      // ... + Q0, then -1/2
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
//   minimax polynomial of exp r up to r^11 (trig_coefficients.py: < 2e-17 relative);  result = p 2^k, the scaling done as two
//   multiplications by 2^(k/2) so that overflow gives inf and underflow goes through the subnormals to 0.
// Relative error <= 2.5e-16 against long-double exp on |x| <= 700 (tests/test_host_logic.py); x is clamped to
// [-750, 750] first (exp(-750) = 0, exp(750) = inf in fp64 anyway); NaN in, NaN out (a select).
#define EXP_CW_COEFS                                                                                         \
    { 1.4426950408889634 /* log2 e */, 0.6931471805599453 /* ln2 hi */, 2.3190468138462996e-17 /* ln2 lo */, \
      /* exp r = 1 + r + r^2 E(r), coefficients of r^11 ... r^2 (trig_coefficients.py) */                    \
      2.511003917993252e-08, 2.7620076799169895e-07, 2.755724236484932e-06, 2.4801521320156154e-05,          \
      0.00019841269886566399, 0.0013888888917198386, 0.008333333333322215, 0.04166666666662416,           \
      0.16666666666666674, 0.5000000000000001 }
#if defined(__CUDACC__)
static __constant__ double exp_cw_dev[13] = EXP_CW_COEFS;
#endif
static const double exp_cw_host[13] = EXP_CW_COEFS;

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
    for (int i = 4; i <= 12; ++i) p = fma(p, r, K[i]);       // E(r)
    p = fma(p * r, r, r) + 1.0;                              // 1 + r + r^2 E(r)
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
