// Host build of the product's branch-free sin/cos (paper_1601_04640_b200/csrc/trig.cuh) so that a
// CPU test can pin it against libm.  Compiled by tests/test_host_logic.py with g++; not part of libdbec.so.
#include <cmath>
#include "../paper_1601_04640_b200/csrc/trig.cuh"
extern "C" void sincos_cw_array(const double* u, double* sn, double* cs, long n) {
    for (long i = 0; i < n; ++i) sincos_cw(u[i], sn + i, cs + i);
}
