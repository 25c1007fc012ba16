// cplx.cuh — complex128 helpers for the dipolar SSCN kernels (product path; shares nothing with oracle/).
#pragma once

#if defined(__CUDACC__)
#define DBEC_HD __host__ __device__ __forceinline__
#else
#define DBEC_HD inline
#endif

#if !defined(__CUDACC__)
struct alignas(16) double2 { double x, y; };
#endif

typedef double2 cd;   // (re, im), 16-byte aligned: one LDG.128 / STG.128 / LDS.128 per element

DBEC_HD cd cmake(double x, double y) { cd r; r.x = x; r.y = y; return r; }
DBEC_HD cd cadd(cd a, cd b) { return cmake(a.x + b.x, a.y + b.y); }
DBEC_HD cd csub(cd a, cd b) { return cmake(a.x - b.x, a.y - b.y); }
DBEC_HD cd cmul(cd a, cd b) { return cmake(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
DBEC_HD cd cmul(double a, cd b) { return cmake(a * b.x, a * b.y); }
DBEC_HD cd cmulc(cd a, cd b) { /* a * conj(b) */ return cmake(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
DBEC_HD cd cconj(cd a) { return cmake(a.x, -a.y); }
DBEC_HD double cnorm2(cd a) { return a.x * a.x + a.y * a.y; }
// a + b*c
DBEC_HD cd cfma(cd b, cd c, cd a) { return cmake(a.x + b.x * c.x - b.y * c.y, a.y + b.x * c.y + b.y * c.x); }
DBEC_HD cd cfma(double b, cd c, cd a) { return cmake(a.x + b * c.x, a.y + b * c.y); }
// multiply by S*i, S = +1 or -1
template <int S> DBEC_HD cd cmul_si(cd a) { return S > 0 ? cmake(-a.y, a.x) : cmake(a.y, -a.x); }
// twiddle as stored (forward, exp(-i theta)) or conjugated (inverse)
template <int S> DBEC_HD cd tw_dir(cd w) { return S < 0 ? w : cmake(w.x, -w.y); }
