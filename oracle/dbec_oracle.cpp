// dbec_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, fp64 CPU implementation of one split-step semi-implicit Crank-Nicolson (SSCN) time
// step of the 2-D/3-D dipolar Gross-Pitaevskii equation, written from the paper text
// (/root/reference/PAPER.md, arxiv 1601.04640) under the readings S1..S24 listed in DESIGN.md
// (PAPER.md prints no formula; every constant below is a stated reading).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this library.  It shares no code with the CUDA path (paper_1601_04640_b200/csrc): own
// struct declarations, own FFT, own Thomas solve, own tables.  The product never calls it.
//
// What each function follows:
//   * oracle_fft_*            PAPER.md:63 "Fourier transformation to momentum space" — the DFT by
//                             its definition (S7, S8), evaluated by a textbook iterative radix-2
//                             FFT whose twiddles come from cos/sin of the exact angle (powers of two)
//                             or by a textbook recursive Cooley-Tukey over the prime factors (any other
//                             length); a separate O(N^2) sum (oracle_dft_naive_*)
//                             pins both.
//   * oracle_vdd3d / _vdd2d   PAPER.md:63, :75 (`potdd`) under readings S3, S4, S5, S6, S21; _vdd2d_xz:
//                             the in-plane-dipole kernel of the 2dXZ programs, reading S25.
//   * oracle_phi_dd           PAPER.md:63, :71 (`calcpsidd2`): n -> DFT -> x V_dd -> inverse DFT.
//                             Plain complex-to-complex transforms of the full grid; the paper's
//                             R2C/C2R trick (:71) is an optimisation that reaches the same numbers.
//   * oracle_nonlinear        PAPER.md:67 (`calcnu`), reading S1/S10 (BASELINE.json part (2)).
//   * oracle_cn_sweep         PAPER.md:67, :79 (`calclux/y/z`, "recursive relation"): textbook
//                             Thomas elimination on every grid line, readings S11, S12.
//   * oracle_normalize        PAPER.md:67 (`calcnorm`), reading S13.
//   * oracle_observables      PAPER.md:67, :71 (`calcmuen`, `calcrms`), readings S13..S16.
//   * dbec_oracle_step        the order nonlinear -> x -> y -> z -> norm (reading S10).
//   * dbec_oracle_set_ramp    PAPER.md:157, :173, :191 ("NSTP"): linear ramp of G and D over the first
//                             NSTP steps, reading S26.
//   * dbec_oracle_density_*   PAPER.md:69 (output of the wave function): integrated 1-D / 2-D densities,
//                             reading S27.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): naive DFT, Parseval, dense tridiagonal solve,
// sine-mode closed form, sampled-Gaussian closed forms, V_dd symmetries, Gaussian dipolar-energy
// closed form, non-interacting ground-state energy, real-time norm conservation, a numpy/scipy
// library restatement.  Nothing here is "parity unpinned".
//
// Parallelism: OpenMP over independent grid lines / points only.  Reductions are accumulated in
// long double in a fixed order (per line, then over lines) so results do not depend on the thread
// count.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;

extern "C" {

// Same field order as the product's dbec_params, declared again on purpose (no shared header).
typedef struct {
    int32_t ndim;       // 2 or 3
    int32_t plane;      // 2-D only: 0 = XY (dipoles along the frozen z), 1 = XZ (dipoles in the plane, S25)
    int32_t nx, ny, nz; // nz = 1 in 2-D
    double dx, dy, dz;
    double dt;
    double nu, lambda, kappa; // V = 1/2 (nu^2 x^2 + lambda^2 y^2 + kappa^2 z^2)   (S2)
    double G, D;              // coefficients of |psi|^2 and Phi_dd                 (S3)
    double d_perp;            // 2-D: width of the frozen direction                 (S21)
    double cutoff;            // 3-D: spherical truncation radius R, 0 = none       (S5)
    int32_t time_mode;        // 0 imaginary, 1 real
} oracle_params;

typedef struct {
    double norm, mu, energy, rms_x, rms_y, rms_z, rms_r, density0, density_max;
} oracle_obs;

struct oracle_state {
    oracle_params p;
    std::vector<cplx> psi;
    std::vector<double> vdd;   // V_dd(k) on the full index grid, built once (PAPER.md:75 `potdd`)
    // S26: ramp of the nonlinear coefficients over the first NSTP steps ("NSTP")
    int ramp_n = 0, ramp_k = 0;
    double G0 = 0, D0 = 0, G1 = 0, D1 = 0;
};

} // extern "C"

static const double PI = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------------------------
// DFT (S7, S8): X[m] = sum_j x[j] exp(sign * 2 pi i m j / N), sign = -1 forward, +1 inverse,
// no scaling in either direction (the 1/P of the inverse is applied by the caller).
// ---------------------------------------------------------------------------------------------

// O(N^2) definition, used only to pin the FFT on tiny inputs.
static void dft_naive_line(const cplx* in, cplx* out, int n, int sign) {
    for (int m = 0; m < n; ++m) {
        long double sr = 0.0L, si = 0.0L;
        for (int j = 0; j < n; ++j) {
            // reduce m*j mod n first so that the angle is exact to rounding of one product
            long long mj = ((long long)m * j) % n;
            long double ang = (long double)sign * 2.0L * 3.14159265358979323846264338327950288L *
                              (long double)mj / (long double)n;
            long double c = cosl(ang), s = sinl(ang);
            sr += (long double)in[j].real() * c - (long double)in[j].imag() * s;
            si += (long double)in[j].real() * s + (long double)in[j].imag() * c;
        }
        out[m] = cplx((double)sr, (double)si);
    }
}

// Textbook iterative radix-2 decimation-in-time FFT, in place, n a power of two.
// tw[k] = exp(sign 2 pi i k / n), k < n/2, each from cos/sin of its own angle (no recurrence).
static void fft_radix2_line(cplx* a, int n, const cplx* tw) {
    // bit reversal
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(a[i], a[j]);
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int i = 0; i < n; i += len) {
            for (int k = 0; k < half; ++k) {
                cplx w = tw[k * step];
                cplx u = a[i + k];
                cplx v = cplx(a[i + k + half].real() * w.real() - a[i + k + half].imag() * w.imag(),
                              a[i + k + half].real() * w.imag() + a[i + k + half].imag() * w.real());
                a[i + k] = u + v;
                a[i + k + half] = u - v;
            }
        }
    }
}

static bool is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }

// Textbook recursive Cooley-Tukey for ANY length (the paper's grids are mostly not
// powers of two): n = p m with p the smallest prime factor of n,
//   X[k + q m] = sum_{r < p} W_n^{r (k + q m)} Y_r[k],   Y_r = DFT_m of the samples r, r + p, r + 2p, ...
// and a prime length straight from the definition.  root[j] = exp(sign 2 pi i j / nroot), nroot a multiple of n,
// each entry from cos/sin of its own angle.  `in` is read with the given stride, `out` is contiguous.
static void fft_any_rec(const cplx* in, long long stride, cplx* out, int n, const cplx* root, int nroot, cplx* work) {
    if (n == 1) { out[0] = in[0]; return; }
    int p = n;
    for (int f = 2; (long long)f * f <= n; ++f) if (n % f == 0) { p = f; break; }
    const int step = nroot / n;                    // W_n^j = root[j * step]
    if (p == n) {                                  // prime: the definition
        for (int k = 0; k < n; ++k) {
            cplx acc(0.0, 0.0);
            for (int j = 0; j < n; ++j) acc += in[j * stride] * root[(((long long)j * k) % n) * step];
            out[k] = acc;
        }
        return;
    }
    const int m = n / p;
    // Y_r into work[r*m .. r*m + m), recursion scratch behind it
    for (int r = 0; r < p; ++r) fft_any_rec(in + r * stride, stride * p, work + (long long)r * m, m, root, nroot, work + n);
    for (int k = 0; k < m; ++k)
        for (int q = 0; q < p; ++q) {
            cplx acc(0.0, 0.0);
            for (int r = 0; r < p; ++r) acc += work[(long long)r * m + k] * root[(((long long)r * (k + q * m)) % n) * step];
            out[k + q * m] = acc;
        }
}

static std::vector<cplx> make_roots(int n, int sign) {
    std::vector<cplx> root(n);
    for (int j = 0; j < n; ++j) {
        double ang = sign * 2.0 * PI * (double)j / (double)n;
        root[j] = cplx(std::cos(ang), std::sin(ang));
    }
    return root;
}

static std::vector<cplx> make_twiddles(int n, int sign) {
    std::vector<cplx> tw(n / 2 > 0 ? n / 2 : 1);
    for (int k = 0; k < n / 2; ++k) {
        double ang = sign * 2.0 * PI * (double)k / (double)n;
        tw[k] = cplx(std::cos(ang), std::sin(ang));
    }
    return tw;
}

// Transform all lines of a[nz][ny][nx] along `axis` (0 = x fastest, 1 = y, 2 = z).
// naive != 0 uses the O(N^2) definition instead of the FFT.
static int transform_axis(cplx* a, int nx, int ny, int nz, int axis, int sign, int naive) {
    int n = axis == 0 ? nx : axis == 1 ? ny : nz;
    if (n == 1) return 0;
    const bool mixed = !naive && !is_pow2(n);      // lengths with other factors: fft_any_rec
    long long stride = axis == 0 ? 1 : axis == 1 ? nx : (long long)nx * ny;
    int n1 = axis == 0 ? ny : nx;             // inner count of lines
    int n2 = axis == 2 ? ny : nz;             // outer count of lines
    long long s1 = axis == 0 ? nx : 1;        // stride between lines (inner)
    long long s2 = axis == 2 ? nx : (long long)nx * ny; // stride between lines (outer)
    std::vector<cplx> tw = make_twiddles(n, sign);
    std::vector<cplx> root = mixed ? make_roots(n, sign) : std::vector<cplx>();
#pragma omp parallel
    {
        std::vector<cplx> buf(n), out(n), work(mixed ? 2 * (size_t)n + 64 : 1);
#pragma omp for collapse(2) schedule(static)
        for (int o = 0; o < n2; ++o) {
            for (int i = 0; i < n1; ++i) {
                cplx* base = a + o * s2 + i * s1;
                for (int j = 0; j < n; ++j) buf[j] = base[j * stride];
                if (naive) {
                    dft_naive_line(buf.data(), out.data(), n, sign);
                    for (int j = 0; j < n; ++j) base[j * stride] = out[j];
                } else if (mixed) {
                    fft_any_rec(buf.data(), 1, out.data(), n, root.data(), n, work.data());
                    for (int j = 0; j < n; ++j) base[j * stride] = out[j];
                } else {
                    fft_radix2_line(buf.data(), n, tw.data());
                    for (int j = 0; j < n; ++j) base[j * stride] = buf[j];
                }
            }
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Dipolar kernels (S3, S4, S5, S6, S21)
// ---------------------------------------------------------------------------------------------

// S6: k_m = 2 pi mt / (N d), mt = m for m < N/2, m - N otherwise.
static double wavenumber(int m, int n, double d) {
    int mt = (m < n / 2) ? m : m - n;   // for even n the Nyquist index n/2 maps to -n/2
    if (n == 1) mt = 0;
    return 2.0 * PI * (double)mt / ((double)n * d);
}

// erfcx(x) = exp(x^2) erfc(x) for x >= 0, stable for large x (S21).
// x < 3: the product itself (both factors are well inside range);
// x >= 3: Laplace continued fraction  sqrt(pi) erfcx(x) = 1/(x+ (1/2)/(x+ 1/(x+ (3/2)/(x+ ...)))),
// evaluated bottom-up with a fixed depth (converges geometrically for x >= 3).
static double erfcx_pos(double x) {
    if (x < 3.0) return std::exp(x * x) * std::erfc(x);
    long double xl = x, f = xl;
    for (int k = 400; k >= 1; --k) f = xl + (0.5L * k) / f;
    return (double)(1.0L / (f * 1.77245385090551602729816748334114518L));
}

static double vdd3d(double kx, double ky, double kz, double cutoff) {
    double k2 = kx * kx + ky * ky + kz * kz;
    if (k2 == 0.0) return 0.0;                               // S4
    double v = 3.0 * kz * kz / k2 - 1.0;                     // S3: 3 cos^2(theta_k) - 1
    if (cutoff > 0.0) {                                      // S5: spherical truncation at R
        double kr = std::sqrt(k2) * cutoff;
        v *= 1.0 + 3.0 * std::cos(kr) / (kr * kr) - 3.0 * std::sin(kr) / (kr * kr * kr);
    }
    return v;
}

static double vdd2d(double kx, double ky, double d_perp) {
    double xi = std::sqrt(kx * kx + ky * ky) * d_perp / std::sqrt(2.0);
    return 2.0 - 3.0 * std::sqrt(PI) * xi * erfcx_pos(xi);   // S21
}

// S25 (the imag2dXZ / real2dXZ programs): 2-D in the x-z plane, the
// dipoles (along z) lie IN the plane and y is the frozen Gaussian direction of width d_perp.  The 3-D
// kernel averaged over k_y with the weight of that Gaussian,
//   int dk_y  d/sqrt(2 pi) exp(-k_y^2 d^2 / 2) (3 k_z^2 / (k_x^2 + k_y^2 + k_z^2) - 1)
//     = -1 + 3 sqrt(pi) (xi_z^2 / xi) erfcx(xi),   xi = sqrt(k_x^2 + k_z^2) d/sqrt(2),  xi_z = k_z d/sqrt(2);
// at k = 0 the second term vanishes (xi_z^2 <= xi^2): value -1.
static double vdd2d_xz(double kx, double kz, double d_perp) {
    double xi = std::sqrt(kx * kx + kz * kz) * d_perp / std::sqrt(2.0);
    if (xi == 0.0) return -1.0;
    double xiz = kz * d_perp / std::sqrt(2.0);
    return -1.0 + 3.0 * std::sqrt(PI) * (xiz * xiz / xi) * erfcx_pos(xi);
}

static double vdd_at(const oracle_params& p, int mx, int my, int mz) {
    double kx = wavenumber(mx, p.nx, p.dx), ky = wavenumber(my, p.ny, p.dy);
    // 2-D XZ: the second grid axis (ny, dy) IS the z axis
    if (p.ndim == 2 && p.plane == 1) return vdd2d_xz(kx, ky, p.d_perp);
    if (p.ndim == 2) return vdd2d(kx, ky, p.d_perp);
    return vdd3d(kx, ky, wavenumber(mz, p.nz, p.dz), p.cutoff);
}

// ---------------------------------------------------------------------------------------------
// Steps of the method
// ---------------------------------------------------------------------------------------------

static long long npoints(const oracle_params& p) { return (long long)p.nx * p.ny * p.nz; }
static double cell_volume(const oracle_params& p) { return p.ndim == 2 ? p.dx * p.dy : p.dx * p.dy * p.dz; }
static double coord(int i, int n, double d) { return (double)(i - n / 2) * d; }   // S17

static int check_params(const oracle_params* p) {
    if (!p) return -1;
    if (p->ndim != 2 && p->ndim != 3) return -1;
    if (p->plane != 0 && !(p->ndim == 2 && p->plane == 1)) return -1;
    if (p->nx < 2 || p->ny < 2 || p->nz < 1) return -1;
    if (p->ndim == 2 && p->nz != 1) return -1;
    if (p->ndim == 3 && p->nz < 2) return -1;
    if (!(p->dx > 0) || !(p->dy > 0) || !(p->dt > 0)) return -1;
    if (p->ndim == 3 && !(p->dz > 0)) return -1;
    if (p->time_mode != 0 && p->time_mode != 1) return -1;
    return 0;
}

// Algorithm steps 1-3: Phi = Re[ (1/P) DFT^-1( V_dd(k) DFT(n) ) ]   (S8, S9)
static void build_vdd(const oracle_params& p, double* out) {
#pragma omp parallel for collapse(2) schedule(static)
    for (int mz = 0; mz < p.nz; ++mz)
        for (int my = 0; my < p.ny; ++my)
            for (int mx = 0; mx < p.nx; ++mx)
                out[mx + (long long)p.nx * (my + (long long)p.ny * mz)] = vdd_at(p, mx, my, mz);
}

static int phi_dd(const oracle_params& p, const double* vdd, const double* dens, double* phi, int naive) {
    long long P = npoints(p);
    std::vector<cplx> w(P);
    for (long long i = 0; i < P; ++i) w[i] = cplx(dens[i], 0.0);
    for (int ax = 0; ax < 3; ++ax)
        if (transform_axis(w.data(), p.nx, p.ny, p.nz, ax, -1, naive)) return -2;
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < P; ++i) w[i] *= vdd[i];
    for (int ax = 0; ax < 3; ++ax)
        if (transform_axis(w.data(), p.nx, p.ny, p.nz, ax, +1, naive)) return -2;
    double invP = 1.0 / (double)P;
    for (long long i = 0; i < P; ++i) phi[i] = w[i].real() * invP;
    return 0;
}

// Algorithm step 4: psi_j <- psi_j exp(-c dt (V_j + G n_j + D Phi_j)), c = 1 or i.
static void nonlinear(const oracle_params& p, cplx* psi, const double* phi) {
#pragma omp parallel for collapse(2) schedule(static)
    for (int iz = 0; iz < p.nz; ++iz)
        for (int iy = 0; iy < p.ny; ++iy)
            for (int ix = 0; ix < p.nx; ++ix) {
                long long i = ix + (long long)p.nx * (iy + (long long)p.ny * iz);
                double x = coord(ix, p.nx, p.dx), y = coord(iy, p.ny, p.dy);
                double z = p.ndim == 3 ? coord(iz, p.nz, p.dz) : 0.0;
                double V = 0.5 * (p.nu * p.nu * x * x + p.lambda * p.lambda * y * y + p.kappa * p.kappa * z * z);
                double n = std::norm(psi[i]);
                double u = p.dt * (V + p.G * n + p.D * phi[i]);
                if (p.time_mode == 0) psi[i] *= std::exp(-u);
                else psi[i] *= cplx(std::cos(u), -std::sin(u));
            }
}

// Textbook Thomas algorithm for the constant tridiagonal system
//   e u_{j-1} + b u_j + e u_{j+1} = r_j,  j = 1..M,  u_0 = u_{M+1} = 0.
// r and u are 1-based views of length M (r[0..M-1]); c, d are scratch of length M.
static void thomas_const(int M, cplx e, cplx b, const cplx* r, cplx* u, cplx* c, cplx* d) {
    c[0] = e / b;
    d[0] = r[0] / b;
    for (int j = 1; j < M; ++j) {
        cplx den = b - e * c[j - 1];
        c[j] = e / den;
        d[j] = (r[j] - e * d[j - 1]) / den;
    }
    u[M - 1] = d[M - 1];
    for (int j = M - 2; j >= 0; --j) u[j] = d[j] - c[j] * u[j + 1];
}

// Algorithm step 5 on one line of N points (in place): Crank-Nicolson with a = c dt / (4 h^2),
// homogeneous Dirichlet ends (S11).
static void cn_line(cplx* line, int N, cplx a, cplx* r, cplx* u, cplx* c, cplx* d) {
    int M = N - 2;
    if (M >= 1) {
        for (int j = 1; j <= M; ++j)
            r[j - 1] = a * line[j - 1] + (1.0 - 2.0 * a) * line[j] + a * line[j + 1];
        thomas_const(M, -a, 1.0 + 2.0 * a, r, u, c, d);
        for (int j = 1; j <= M; ++j) line[j] = u[j - 1];
    }
    line[0] = 0.0;
    line[N - 1] = 0.0;
}

static void cn_sweep(const oracle_params& p, cplx* psi, int axis) {
    int nx = p.nx, ny = p.ny, nz = p.nz;
    int n = axis == 0 ? nx : axis == 1 ? ny : nz;
    if (n == 1) return;
    double h = axis == 0 ? p.dx : axis == 1 ? p.dy : p.dz;
    double ar = p.dt / (4.0 * h * h);
    cplx a = p.time_mode == 0 ? cplx(ar, 0.0) : cplx(0.0, ar);
    long long stride = axis == 0 ? 1 : axis == 1 ? nx : (long long)nx * ny;
    int n1 = axis == 0 ? ny : nx;
    int n2 = axis == 2 ? ny : nz;
    long long s1 = axis == 0 ? nx : 1;
    long long s2 = axis == 2 ? nx : (long long)nx * ny;
#pragma omp parallel
    {
        std::vector<cplx> buf(n), r(n), u(n), c(n), d(n);
#pragma omp for collapse(2) schedule(static)
        for (int o = 0; o < n2; ++o)
            for (int i = 0; i < n1; ++i) {
                cplx* base = psi + o * s2 + i * s1;
                for (int j = 0; j < n; ++j) buf[j] = base[j * stride];
                cn_line(buf.data(), n, a, r.data(), u.data(), c.data(), d.data());
                for (int j = 0; j < n; ++j) base[j * stride] = buf[j];
            }
    }
}

// Sum over the whole grid of f(i), long double, fixed order: per x-line, then over lines.
template <class F>
static long double grid_sum(const oracle_params& p, F f) {
    int lines = p.ny * p.nz;
    std::vector<long double> part(lines);
#pragma omp parallel for schedule(static)
    for (int l = 0; l < lines; ++l) {
        long double s = 0.0L;
        int iy = l % p.ny, iz = l / p.ny;
        for (int ix = 0; ix < p.nx; ++ix) s += f(ix, iy, iz);
        part[l] = s;
    }
    long double tot = 0.0L;
    for (int l = 0; l < lines; ++l) tot += part[l];
    return tot;
}

static double norm_integral(const oracle_params& p, const cplx* psi) {
    long double s = grid_sum(p, [&](int ix, int iy, int iz) -> long double {
        long long i = ix + (long long)p.nx * (iy + (long long)p.ny * iz);
        return (long double)psi[i].real() * psi[i].real() + (long double)psi[i].imag() * psi[i].imag();
    });
    return (double)(s * (long double)cell_volume(p));   // S13
}

// Algorithm step 6.
static void normalize(const oracle_params& p, cplx* psi) {
    double S = norm_integral(p, psi);
    double f = 1.0 / std::sqrt(S);
    long long P = npoints(p);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < P; ++i) psi[i] *= f;
}

static int one_step(const oracle_params& p, const double* vdd, cplx* psi) {
    long long P = npoints(p);
    std::vector<double> dens(P), phi(P);
    for (long long i = 0; i < P; ++i) dens[i] = std::norm(psi[i]);
    int rc = phi_dd(p, vdd, dens.data(), phi.data(), 0);
    if (rc) return rc;
    nonlinear(p, psi, phi.data());
    cn_sweep(p, psi, 0);
    cn_sweep(p, psi, 1);
    cn_sweep(p, psi, 2);
    if (p.time_mode == 0) normalize(p, psi);
    return 0;
}

static int observables(const oracle_params& p, const double* vdd, const cplx* psi, oracle_obs* o) {
    long long P = npoints(p);
    int nx = p.nx, ny = p.ny, nz = p.nz;
    std::vector<double> dens(P), phi(P);
    for (long long i = 0; i < P; ++i) dens[i] = std::norm(psi[i]);
    int rc = phi_dd(p, vdd, dens.data(), phi.data(), 0);
    if (rc) return rc;
    long double dV = cell_volume(p);
    auto at = [&](int ix, int iy, int iz) { return ix + (long long)nx * (iy + (long long)ny * iz); };
    long double S = grid_sum(p, [&](int ix, int iy, int iz) -> long double { return dens[at(ix, iy, iz)]; }) * dV;
    // S14: forward differences across every link, per direction
    long double ekx = grid_sum(p, [&](int ix, int iy, int iz) -> long double {
        if (ix + 1 >= nx) return 0.0L;
        cplx d = psi[at(ix + 1, iy, iz)] - psi[at(ix, iy, iz)];
        return (long double)d.real() * d.real() + (long double)d.imag() * d.imag();
    });
    long double eky = grid_sum(p, [&](int ix, int iy, int iz) -> long double {
        if (iy + 1 >= ny) return 0.0L;
        cplx d = psi[at(ix, iy + 1, iz)] - psi[at(ix, iy, iz)];
        return (long double)d.real() * d.real() + (long double)d.imag() * d.imag();
    });
    long double ekz = 0.0L;
    if (p.ndim == 3)
        ekz = grid_sum(p, [&](int ix, int iy, int iz) -> long double {
            if (iz + 1 >= nz) return 0.0L;
            cplx d = psi[at(ix, iy, iz + 1)] - psi[at(ix, iy, iz)];
            return (long double)d.real() * d.real() + (long double)d.imag() * d.imag();
        });
    long double ekin = 0.5L * dV * (ekx / ((long double)p.dx * p.dx) + eky / ((long double)p.dy * p.dy) +
                                    (p.ndim == 3 ? ekz / ((long double)p.dz * p.dz) : 0.0L));
    long double sx2 = grid_sum(p, [&](int ix, int iy, int iz) -> long double {
        long double x = coord(ix, nx, p.dx); return x * x * dens[at(ix, iy, iz)]; }) * dV;
    long double sy2 = grid_sum(p, [&](int ix, int iy, int iz) -> long double {
        long double y = coord(iy, ny, p.dy); return y * y * dens[at(ix, iy, iz)]; }) * dV;
    long double sz2 = 0.0L;
    if (p.ndim == 3)
        sz2 = grid_sum(p, [&](int ix, int iy, int iz) -> long double {
            long double z = coord(iz, nz, p.dz); return z * z * dens[at(ix, iy, iz)]; }) * dV;
    long double etr = 0.5L * ((long double)p.nu * p.nu * sx2 + (long double)p.lambda * p.lambda * sy2 +
                              (long double)p.kappa * p.kappa * sz2);
    long double ec = (long double)p.G * dV * grid_sum(p, [&](int ix, int iy, int iz) -> long double {
        long double n = dens[at(ix, iy, iz)]; return n * n; });
    long double ed = (long double)p.D * dV * grid_sum(p, [&](int ix, int iy, int iz) -> long double {
        return (long double)phi[at(ix, iy, iz)] * dens[at(ix, iy, iz)]; });
    o->norm = (double)S;
    o->mu = (double)((ekin + etr + ec + ed) / S);
    o->energy = (double)((ekin + etr + 0.5L * ec + 0.5L * ed) / S);
    o->rms_x = (double)sqrtl(sx2 / S);
    o->rms_y = (double)sqrtl(sy2 / S);
    o->rms_z = (double)sqrtl(sz2 / S);
    o->rms_r = (double)sqrtl((sx2 + sy2 + sz2) / S);
    o->density0 = dens[at(nx / 2, ny / 2, p.ndim == 3 ? nz / 2 : 0)];
    double dmax = 0.0;
    for (long long i = 0; i < P; ++i) dmax = dens[i] > dmax ? dens[i] : dmax;
    o->density_max = dmax;
    return 0;
}

// ---------------------------------------------------------------------------------------------
// C ABI (host memory everywhere)
// ---------------------------------------------------------------------------------------------
extern "C" {

int dbec_oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int dbec_oracle_create(const oracle_params* p, oracle_state** out) {
    int rc = check_params(p);
    if (rc) return rc;
    if (!out) return -1;
    oracle_state* s = new oracle_state;
    s->p = *p;
    s->psi.assign(npoints(*p), cplx(0.0, 0.0));
    s->vdd.resize(npoints(*p));
    build_vdd(s->p, s->vdd.data());
    *out = s;
    return 0;
}

int dbec_oracle_destroy(oracle_state* s) { delete s; return 0; }

int dbec_oracle_set_psi(oracle_state* s, const double* psi_c128) {
    if (!s || !psi_c128) return -1;
    std::memcpy((void*)s->psi.data(), psi_c128, sizeof(cplx) * s->psi.size());
    return 0;
}

int dbec_oracle_get_psi(oracle_state* s, double* psi_c128) {
    if (!s || !psi_c128) return -1;
    std::memcpy(psi_c128, (const void*)s->psi.data(), sizeof(cplx) * s->psi.size());
    return 0;
}

int dbec_oracle_set_coupling(oracle_state* s, double G, double D) {   // S18
    if (!s) return -1;
    s->p.G = G; s->p.D = D;
    s->ramp_n = s->ramp_k = 0;                                        // an explicit value ends any ramp
    return 0;
}

// S26: the k-th step after this call (k = 1..nstp) runs with G0 + (G1 - G0) k/nstp and
// D0 + (D1 - D0) k/nstp; every later step with (G1, D1).  nstp = 0: (G1, D1) at once.
int dbec_oracle_set_ramp(oracle_state* s, int nstp, double G0, double D0, double G1, double D1) {
    if (!s || nstp < 0) return -1;
    s->ramp_n = nstp; s->ramp_k = 0;
    s->G0 = G0; s->D0 = D0; s->G1 = G1; s->D1 = D1;
    if (nstp == 0) { s->p.G = G1; s->p.D = D1; }
    else { s->p.G = G0; s->p.D = D0; }
    return 0;
}

int dbec_oracle_get_coupling(oracle_state* s, double* G, double* D) {
    if (!s || !G || !D) return -1;
    *G = s->p.G; *D = s->p.D;
    return 0;
}

// S27: integrated densities (the lineage's 1-D / 2-D density output, "wave function array is
// returned back to CPU when it is required for writing output"): |psi|^2 summed over the other axes
// times their spacings (plain sums, S13).
//   1-D, axis a:           out[i_a]            = prod_{b != a} d_b  sum_{other indices} |psi|^2
//   2-D, integrated axis a (3-D grids only): out over the two remaining axes, the lower axis fastest
//                          (a = 2: [ny][nx], a = 1: [nz][nx], a = 0: [nz][ny]),  = d_a sum_{i_a} |psi|^2
int dbec_oracle_density_1d(oracle_state* s, int axis, double* out) {
    if (!s || !out || axis < 0 || axis >= s->p.ndim) return -1;
    const oracle_params& p = s->p;
    const int n[3] = {p.nx, p.ny, p.nz};
    const double d[3] = {p.dx, p.dy, p.ndim == 3 ? p.dz : 1.0};
    long double w = 1.0L;
    for (int b = 0; b < p.ndim; ++b) if (b != axis) w *= d[b];
    std::vector<long double> acc(n[axis], 0.0L);
    for (int iz = 0; iz < p.nz; ++iz)
        for (int iy = 0; iy < p.ny; ++iy)
            for (int ix = 0; ix < p.nx; ++ix) {
                const int idx[3] = {ix, iy, iz};
                const cplx v = s->psi[ix + (long long)p.nx * (iy + (long long)p.ny * iz)];
                acc[idx[axis]] += (long double)v.real() * v.real() + (long double)v.imag() * v.imag();
            }
    for (int i = 0; i < n[axis]; ++i) out[i] = (double)(acc[i] * w);
    return 0;
}

int dbec_oracle_density_2d(oracle_state* s, int axis, double* out) {
    if (!s || !out || s->p.ndim != 3 || axis < 0 || axis > 2) return -1;
    const oracle_params& p = s->p;
    const int n[3] = {p.nx, p.ny, p.nz};
    const double d[3] = {p.dx, p.dy, p.dz};
    const int lo = axis == 0 ? 1 : 0, hi = axis == 2 ? 1 : 2;          // the two axes that remain
    std::vector<long double> acc((size_t)n[lo] * n[hi], 0.0L);
    for (int iz = 0; iz < p.nz; ++iz)
        for (int iy = 0; iy < p.ny; ++iy)
            for (int ix = 0; ix < p.nx; ++ix) {
                const int idx[3] = {ix, iy, iz};
                const cplx v = s->psi[ix + (long long)p.nx * (iy + (long long)p.ny * iz)];
                acc[idx[lo] + (size_t)n[lo] * idx[hi]] += (long double)v.real() * v.real() + (long double)v.imag() * v.imag();
            }
    for (size_t i = 0; i < acc.size(); ++i) out[i] = (double)(acc[i] * (long double)d[axis]);
    return 0;
}

int dbec_oracle_step(oracle_state* s, int nsteps) {
    if (!s || nsteps < 0) return -1;
    for (int i = 0; i < nsteps; ++i) {
        if (s->ramp_k < s->ramp_n) {                                  // S26
            s->ramp_k += 1;
            const double f = (double)s->ramp_k / (double)s->ramp_n;
            s->p.G = s->G0 + (s->G1 - s->G0) * f;
            s->p.D = s->D0 + (s->D1 - s->D0) * f;
        }
        int rc = one_step(s->p, s->vdd.data(), s->psi.data());
        if (rc) return rc;
    }
    return 0;
}

int dbec_oracle_observables(oracle_state* s, oracle_obs* o) {
    if (!s || !o) return -1;
    return observables(s->p, s->vdd.data(), s->psi.data(), o);
}

// ---- single parts, exported so that each can be pinned and compared on its own ----

// In-place DFT of a[nz][ny][nx] over every axis of length > 1; sign -1 forward, +1 inverse (unscaled).
int dbec_oracle_fft(double* a_c128, int nx, int ny, int nz, int sign, int naive) {
    if (!a_c128 || (sign != 1 && sign != -1)) return -1;
    for (int ax = 0; ax < 3; ++ax)
        if (transform_axis((cplx*)a_c128, nx, ny, nz, ax, sign, naive)) return -2;
    return 0;
}

double dbec_oracle_erfcx(double x) { return erfcx_pos(x); }
double dbec_oracle_vdd3d(double kx, double ky, double kz, double cutoff) { return vdd3d(kx, ky, kz, cutoff); }
double dbec_oracle_vdd2d(double kx, double ky, double d_perp) { return vdd2d(kx, ky, d_perp); }
double dbec_oracle_vdd2d_xz(double kx, double kz, double d_perp) { return vdd2d_xz(kx, kz, d_perp); }
double dbec_oracle_wavenumber(int m, int n, double d) { return wavenumber(m, n, d); }

// V_dd on the full index grid [nz][ny][nx].
int dbec_oracle_vdd_table(const oracle_params* p, double* out) {
    if (!p || !out) return -1;
    build_vdd(*p, out);
    return 0;
}

int dbec_oracle_phi_dd(const oracle_params* p, const double* dens, double* phi, int naive) {
    if (!p || !dens || !phi) return -1;
    if (!naive && check_params(p)) return -2;
    std::vector<double> vdd(npoints(*p));
    build_vdd(*p, vdd.data());
    return phi_dd(*p, vdd.data(), dens, phi, naive);
}

int dbec_oracle_nonlinear(const oracle_params* p, double* psi_c128, const double* phi) {
    if (check_params(p) || !psi_c128 || !phi) return -1;
    nonlinear(*p, (cplx*)psi_c128, phi);
    return 0;
}

int dbec_oracle_cn_sweep(const oracle_params* p, double* psi_c128, int axis) {
    if (check_params(p) || !psi_c128 || axis < 0 || axis > 2) return -1;
    cn_sweep(*p, (cplx*)psi_c128, axis);
    return 0;
}

// One line of N points with a given complex a (any N >= 3; used by the dense-solve pin).
int dbec_oracle_cn_line(double* line_c128, int N, double a_re, double a_im) {
    if (!line_c128 || N < 3) return -1;
    std::vector<cplx> r(N), u(N), c(N), d(N);
    cn_line((cplx*)line_c128, N, cplx(a_re, a_im), r.data(), u.data(), c.data(), d.data());
    return 0;
}

int dbec_oracle_normalize(const oracle_params* p, double* psi_c128) {
    if (check_params(p) || !psi_c128) return -1;
    normalize(*p, (cplx*)psi_c128);
    return 0;
}

double dbec_oracle_norm(const oracle_params* p, const double* psi_c128) {
    return norm_integral(*p, (const cplx*)psi_c128);
}

} // extern "C"
