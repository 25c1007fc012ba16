// Host build of the product's branch-free sin/cos and exp (paper_1601_04640_b200/csrc/trig.cuh) so that a
// CPU test can pin it against libm.  Compiled by tests/test_host_logic.py with g++; not part of libdbec.so.
#include <cmath>
#include "../paper_1601_04640_b200/csrc/trig.cuh"
extern "C" void sincos_cw_array(const double* u, double* sn, double* cs, long n) {
    for (long i = 0; i < n; ++i) sincos_cw(u[i], sn + i, cs + i);
}
extern "C" void exp_cw_array(const double* x, double* e, long n) {
    for (long i = 0; i < n; ++i) e[i] = exp_cw(x[i]);
}
