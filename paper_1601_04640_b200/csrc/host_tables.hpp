// host_tables.hpp — small per-axis tables built on the host at dbec_create time (product path).
//
// FFT twiddles and the Crank-Nicolson coefficients of one axis (the
// per-line "cbeta" array of the paper depends only on (a, N) for a constant-coefficient line, so it
// is one table per axis here instead of one array per thread).
#pragma once
#include <cmath>
#include <complex>
#include <vector>

namespace dbec_host {

typedef std::complex<double> zc;

// twN[j] = exp(-2 pi i j / N), j < N; angles reduced to the first octant in long double.
inline void make_twN(int N, std::vector<zc>& tw) {
    tw.resize(N);
    const long double PI = 3.14159265358979323846264338327950288L;
    for (int j = 0; j < N; ++j) {
        long double ang = 2.0L * PI * (long double)j / (long double)N;
        tw[j] = zc((double)cosl(ang), (double)(-sinl(ang)));
    }
    // exact values on the axes
    tw[0] = zc(1.0, 0.0);
    if (N % 2 == 0) tw[N / 2] = zc(-1.0, 0.0);
    if (N % 4 == 0) { tw[N / 4] = zc(0.0, -1.0); tw[3 * N / 4] = zc(0.0, 1.0); }
}

// twA[k1*T + m] = exp(-2 pi i m k1 / N), N = 16 T: the stage-1 twiddles in the order the threads read them.
inline void make_twA(int N, const std::vector<zc>& twN, std::vector<zc>& twA) {
    int T = N / 16;
    twA.resize(N);
    for (int k1 = 0; k1 < 16; ++k1)
        for (int m = 0; m < T; ++m) twA[k1 * T + m] = twN[(m * k1) % N];
}

// Crank-Nicolson tables of one axis: h_j, PF_j, PB_j for j < N with chunks of L points.
//   h_0 = h_{N-1} = 0; den_1 = 1+2a; den_j = 1+2a - a h_{j-1}; h_j = a / den_j   (j = 1..N-2)
//   PF_j = prod_{i=j0(j)}^{j} h_i,  PB_j = prod_{i=j}^{jend(j)} h_i  (j0, jend = ends of j's chunk)
inline void make_cn(int N, int L, zc a, std::vector<zc>& h, std::vector<zc>& pf, std::vector<zc>& pb) {
    h.assign(N, zc(0.0, 0.0));
    pf.assign(N, zc(0.0, 0.0));
    pb.assign(N, zc(0.0, 0.0));
    zc b = 1.0 + 2.0 * a;
    for (int j = 1; j <= N - 2; ++j) {
        zc den = b - a * h[j - 1];
        h[j] = a / den;
    }
    for (int j0 = 0; j0 < N; j0 += L) {
        int je = (j0 + L < N ? j0 + L : N) - 1;
        zc p(1.0, 0.0);
        for (int j = j0; j <= je; ++j) { p *= h[j]; pf[j] = p; }
        p = zc(1.0, 0.0);
        for (int j = je; j >= j0; --j) { p *= h[j]; pb[j] = p; }
    }
}

}  // namespace dbec_host
