// trig.cuh — branch-free sin/cos pair for the real-time nonlinear step (calcnu):
// psi <- psi exp(-i u), u = dt (V + G|psi|^2 + D Phi_dd).
//
// The CUDA library sincos carries a slow-path branch for huge arguments; sixteen calls in a row then
// run one after the other.  This version has no branch, so the compiler interleaves the sixteen
// evaluations of a thread (the fp64 pipe has an 8-cycle dependent latency on sm_100a).
//   k = nearest integer to u 2/pi;  r = u - k pi/2 with pi/2 as the sum of three doubles and FMAs
//   (exact to < 1e-19 for |k| < 2^30);  Taylor polynomials of sin r / cos r on |r| <= pi/4 up to
//   r^15 / r^16 (truncation < 5e-17);  quadrant from k mod 4.
// Absolute error <= 1.5e-16 against long-double sin/cos for |u| <= SINCOS_CW_MAX = 1e14 (checked on
// the host by tests/test_host_logic.py; the reduction is exact while |k| < 2^51).  Beyond that, where
// one ulp of u is already a sizeable part of a turn and the time step is meaningless anyway, and for
// non-finite u, both results are NaN (a select, not a branch), as loud as the library's behaviour
// for infinities.
#pragma once
#include "cplx.cuh"

#define SINCOS_CW_MAX 1.0e14

DBEC_HD void sincos_cw(double u, double* sn, double* cs) {
    u = (fabs(u) <= SINCOS_CW_MAX) ? u : (u - u) / (u - u);   // out of range or not finite -> NaN
    const double MAGIC = 6755399441055744.0;                 // 1.5 * 2^52: adding it rounds to nearest integer
    const double kb = u * 0.63661977236758134 + MAGIC;
    const double kd = kb - MAGIC;
#if defined(__CUDA_ARCH__)
    const int q = __double2loint(kb);
#else
    union { double d; unsigned long long u; } cv; cv.d = kb;
    const int q = (int)(unsigned)(cv.u & 0xffffffffull);
#endif
    double r = fma(-kd, 1.5707963267948966, u);
    r = fma(-kd, 6.123233995736766e-17, r);
    r = fma(-kd, -1.4973849048591698e-33, r);
    const double r2 = r * r;
    double ps = -1.0 / 1307674368000.0;                      // -1/15!
    ps = fma(ps, r2, 1.0 / 6227020800.0);                    //  1/13!
    ps = fma(ps, r2, -1.0 / 39916800.0);                     // -1/11!
    ps = fma(ps, r2, 1.0 / 362880.0);                        //  1/9!
    ps = fma(ps, r2, -1.0 / 5040.0);                         // -1/7!
    ps = fma(ps, r2, 1.0 / 120.0);                           //  1/5!
    ps = fma(ps, r2, -1.0 / 6.0);                            // -1/3!
    const double sr = fma(ps * r2, r, r);
    double pc = 1.0 / 20922789888000.0;                      //  1/16!
    pc = fma(pc, r2, -1.0 / 87178291200.0);                  // -1/14!
    pc = fma(pc, r2, 1.0 / 479001600.0);                     //  1/12!
    pc = fma(pc, r2, -1.0 / 3628800.0);                      // -1/10!
    pc = fma(pc, r2, 1.0 / 40320.0);                         //  1/8!
    pc = fma(pc, r2, -1.0 / 720.0);                          // -1/6!
    pc = fma(pc, r2, 1.0 / 24.0);                            //  1/4!
    pc = fma(pc, r2, -0.5);                                  // -1/2!
    const double cr = fma(pc, r2, 1.0);
    const double a = (q & 1) ? cr : sr;                      // sin u up to sign
    const double b = (q & 1) ? sr : cr;                      // cos u up to sign
    *sn = (q & 2) ? -a : a;
    *cs = ((q + 1) & 2) ? -b : b;
}
