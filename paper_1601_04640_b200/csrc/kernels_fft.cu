// kernels_fft.cu — the dipolar mean field (calcpsidd2) and the nonlinear
// step (calcnu) as hand-written sm_100a kernels.  No library FFT.
//
//   k_density_fftx   a1, x axis: n = |s psi|^2 fused into a forward real-to-complex transform.  Two
//                    real grid lines ride one complex FFT (re = line y, im = line y+1) and are split
//                    by Hermitian symmetry ("density ... purely real ... Hermitian").
//   k_fft_strided    a1/a3 along y or z on the half spectrum: tiles of 8 columns x N rows held in
//                    registers, 128-byte coalesced rows.  MODE_FMI chains forward transform, the
//                    multiply by V_dd(k)/P (a2, PAPER.md:63 "convolution theorem", :75 `potdd`) and
//                    the inverse transform of the same axis while the line stays on chip.
//   k_ifftx_nonlin   a3 x axis (complex-to-real, two lines per FFT) fused with
//                    psi <- s psi exp(-c dt (V + G n + D Phi))   (a4), optionally followed by the
//                    Crank-Nicolson sweep along x on the same line (a5), or writing Phi_dd only.
#include "dbec_internal.hpp"
#include "fft_line.cuh"
#include "cn_chunk.cuh"
#include "cn_line_smem.cuh"
#include "tma_pipe.cuh"

template <class P> struct XLine {
    // shared elements per line pair of the contiguous-x kernels: FFT exchange or one padded line
    static constexpr int PADN = P::N + 3 * P::T;   // padded line + two rows of chunk ends (cn_line_smem.cuh)
    static constexpr int SM = (P::SMEM > PADN ? P::SMEM : PADN);
    static constexpr int SMF = (P::SMEM > P::N ? P::SMEM : P::N);   // k_density_fftx: exchange rows or Z[N]
};

// ------------------------------------------------------------------------------------------------
// a1, x axis
// ------------------------------------------------------------------------------------------------
template <class P, int LP>
__global__ void __launch_bounds__(P::T* LP)
k_density_fftx(const cd* __restrict__ psi, cd* __restrict__ spec, const cd* __restrict__ twA,
               const cd* __restrict__ twN, double* __restrict__ scal, int npairs, int nxhp, int pairs_per_member,
               int nb, int advance) {
    extern __shared__ cd smem[];
    pdl_launch_dependents(); pdl_wait();       // (tma_pipe.cuh) launch latency overlaps the previous kernel
    constexpr int T = P::T, N = P::N;
    const int lp = threadIdx.x / T, m = threadIdx.x % T;
    const long long pair = (long long)blockIdx.x * LP + lp;
    const bool active = pair < npairs;
    cd* sm = smem + lp * XLine<P>::SMF;
    const double s2 = scal[(active ? pair / pairs_per_member : 0) * SC_COUNT + SC_S2];
    if (advance && blockIdx.x == 0)            // first kernel of a step: move the NSTP ramp on (reads neither G nor D)
        for (int b = threadIdx.x; b < nb; b += blockDim.x) ramp_advance(scal + (size_t)b * SC_COUNT);
    const cd* pa = psi + (active ? pair : 0) * 2 * N;
    const cd* pb = pa + N;
    cd v[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        cd a = pa[j * T + m], b = pb[j * T + m];
        v[j] = cmake(s2 * cnorm2(a), s2 * cnorm2(b));
    }
    fft_line<P, -1, 0>(v, m, sm, 1, twA, twN);
    __syncwarp();
    // Z[k] to shared memory so that each thread can reach its mirror Z[N-k]
#pragma unroll
    for (int j = 0; j < 16; ++j) sm[j * T + m] = v[j];
    __syncwarp();
    cd* oa = spec + (active ? pair : 0) * 2 * nxhp;
    cd* ob = oa + nxhp;
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const int k = j * T + m;
        if (k <= N / 2) {
            cd z = v[j], zp = sm[(N - k) & (N - 1)];
            // X_a = (Z[k] + conj Z[N-k])/2,  X_b = (Z[k] - conj Z[N-k])/(2i)
            cd xa = cmake(0.5 * (z.x + zp.x), 0.5 * (z.y - zp.y));
            cd xb = cmake(0.5 * (z.y + zp.y), -0.5 * (z.x - zp.x));
            if (active) { oa[k] = xa; ob[k] = xb; }
        } else if (k < nxhp) {
            if (active) { oa[k] = cmake(0.0, 0.0); ob[k] = cmake(0.0, 0.0); }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// strided transforms on the half spectrum
// ------------------------------------------------------------------------------------------------
enum { MODE_FWD = 0, MODE_INV = 1, MODE_FMI = 2 };

// A line's point j sits at  base + j*line_stride,  base = outer*outer_stride + column;  a tile is
// DBEC_SPEC_COLS consecutive columns.  TILES tiles per block.
template <class P, int MODE, int TILES>
__global__ void __launch_bounds__(P::T* DBEC_SPEC_COLS* TILES)
k_fft_strided(cd* __restrict__ spec, const double* __restrict__ vdd, const cd* __restrict__ twA,
              const cd* __restrict__ twN, long long line_stride, long long outer_stride, int ntiles_x,
              long long ntiles, int n, int nxhp, int ny3, long long vdd_line_stride) {
    extern __shared__ cd smem[];
    pdl_launch_dependents(); pdl_wait();
    constexpr int T = P::T, C = DBEC_SPEC_COLS;
    const int tl = threadIdx.x / (T * C), r = threadIdx.x % (T * C);
    const int col = r % C, m = r / C;
    long long tile = (long long)blockIdx.x * TILES + tl;
    const bool active = tile < ntiles;
    if (!active) tile = 0;
    const long long outer = tile / ntiles_x, tx = tile % ntiles_x;
    const long long base = outer * outer_stride + tx * C + col;
    cd* sm = smem + tl * (P::SMEM * C) + col;
    cd* g = spec + base;
    cd v[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = g[(long long)(j * T + m) * line_stride];
    if (MODE == MODE_FWD || MODE == MODE_FMI) fft_line<P, -1, 1>(v, m, sm, C, twA, twN);
    if (MODE == MODE_FMI) {
        // the folded V_dd table (shared by the members of a batch): index r along the line -> min(r, n - r);
        // 3-D (ny3 = NY, lines along z): the tile's columns are (k_y, k_x) flattened, k_y folds the same way
        const long long cix = tx * C + col;
        long long voff = cix;
        if (ny3) { const int ky = (int)(cix / nxhp), kx = (int)(cix % nxhp); voff = (long long)(ky < ny3 - ky ? ky : ny3 - ky) * nxhp + kx; }
        const double* w = vdd + voff;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int r = j * T + m;
            v[j] = cmul(w[(long long)(r < n - r ? r : n - r) * vdd_line_stride], v[j]);
        }
        if (T > 1) __syncthreads();
    }
    if (MODE == MODE_INV || MODE == MODE_FMI) fft_line<P, +1, 1>(v, m, sm, C, twA, twN);
    if (active) {
#pragma unroll
        for (int j = 0; j < 16; ++j) g[(long long)(j * T + m) * line_stride] = v[j];
    }
}

// ------------------------------------------------------------------------------------------------
// a3 (x axis, complex-to-real) + a4 (+ a5)
// ------------------------------------------------------------------------------------------------
enum { NL_STEP = 0, NL_STEP_CNX = 1, NL_PHI = 2 };
#ifndef NL_MINB
#define NL_MINB 4
#endif

template <class P, int LP, bool RT, int MODE>
__global__ void __launch_bounds__(P::T* LP, NL_MINB)
k_ifftx_nonlin(const cd* __restrict__ spec, cd* __restrict__ psi, double* __restrict__ phi_out,
               const cd* __restrict__ twA, const cd* __restrict__ twN, const double* __restrict__ scal,
               const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
               double dt, int npairs, int nxhp, int ny, int nz, CnTab<RT> cn) {
    extern __shared__ cd smem[];
    pdl_launch_dependents(); pdl_wait();
    typedef typename CnCoef<RT>::type CT;
    constexpr int T = P::T, N = P::N;
    const int lp = threadIdx.x / T, m = threadIdx.x % T;
    long long pair = (long long)blockIdx.x * LP + lp;
    const bool active = pair < npairs;
    if (!active) pair = 0;
    CnTab<RT> cs = cn;
    cd* sm = smem + lp * XLine<P>::SM;
    if (MODE == NL_STEP_CNX) {
        cs = cn_stage_tables<RT, N>(cn, (CT*)smem);
        sm += (3 * cn_tab_elems(N) * sizeof(CT)) / sizeof(cd);
    }
    const cd* sa = spec + pair * 2 * nxhp;
    const cd* sb = sa + nxhp;
    cd v[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const int k = j * T + m;
        if (k <= N / 2) {
            cd a = sa[k], b = sb[k];
            v[j] = cmake(a.x - b.y, a.y + b.x);          // X_a + i X_b
        } else {
            cd a = sa[N - k], b = sb[N - k];
            v[j] = cmake(a.x + b.y, b.x - a.y);          // conj X_a + i conj X_b
        }
    }
    if (MODE == NL_STEP_CNX) __syncthreads();            // staged tables visible
    fft_line<P, +1, 0>(v, m, sm, 1, twA, twN);
    // v[j] = (Phi_dd on line y, Phi_dd on line y+1) at x = j*T + m   (1/P is inside the V_dd table)
    if (MODE == NL_PHI) {
        double* fa = phi_out + pair * 2 * N;
        double* fb = fa + N;
        if (active) {
#pragma unroll
            for (int j = 0; j < 16; ++j) { fa[j * T + m] = v[j].x; fb[j * T + m] = v[j].y; }
        }
        return;
    }
    const long long row = pair * 2;
    const int y = (int)(row % ny), zz = (int)(row / ny), z = zz % nz;
    const double* sc = scal + (size_t)(zz / nz) * SC_COUNT;          // this row's batch member
    const double s = sc[SC_S], s2 = sc[SC_S2], G = sc[SC_G], D = sc[SC_D];
    const double vzz = vz[z];
    if (MODE == NL_STEP_CNX) __syncwarp();               // FFT exchange rows are reused by the sweep
#pragma unroll
    for (int l = 0; l < 2; ++l) {
        cd* p = psi + (row + l) * N;
        const double vrow = vy[y + l] + vzz;
        cd q[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) q[j] = p[j * T + m];
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const double phi = l == 0 ? v[j].x : v[j].y;
            const double u = dt * (vx[j * T + m] + vrow + G * (s2 * cnorm2(q[j])) + D * phi);
            if (RT) {
                double sn, cs_;
                sincos(u, &sn, &cs_);
                q[j] = cmul(s, cmul(q[j], cmake(cs_, -sn)));
            } else {
                q[j] = cmul(s * exp(-u), q[j]);
            }
        }
        if (MODE == NL_STEP_CNX) {
            cn_line_via_smem<RT, T, 17>(q, m, sm, cs);
            __syncwarp();
        }
        if (active) {
#pragma unroll
            for (int j = 0; j < 16; ++j) p[j * T + m] = q[j];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// V_dd table (the paper's `potdd`), half spectrum, scaled by 1/P (reading S8)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double wavenumber(int mi, int n, double d) {     // reading S6
    int mt = (mi < n / 2) ? mi : mi - n;
    if (n == 1) mt = 0;
    return 6.283185307179586476925286766559 * (double)mt / ((double)n * d);
}

// Folded: rows m_y = 0..ny/2 and m_z = 0..nz/2 only (the table is even in both; dbec_internal.hpp).
__global__ void k_build_vdd(double* __restrict__ vdd, int ndim, int plane, int nx, int ny, int nz, int nxhp, int nyf, int nzf,
                            double dx, double dy, double dz, double d_perp, double cutoff, double invP) {
    const long long total = (long long)nzf * nyf * nxhp;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        const int mx = (int)(i % nxhp);
        const int my = (int)((i / nxhp) % nyf);
        const int mz = (int)(i / ((long long)nxhp * nyf));
        double v = 0.0;
        if (mx <= nx / 2) {
            const double kx = wavenumber(mx, nx, dx), ky = wavenumber(my, ny, dy);
            if (ndim == 2) {
                const double xi = sqrt(kx * kx + ky * ky) * d_perp * 0.70710678118654752440;
                const double g = 3.0 * 1.7724538509055160272981674833411 * erfcx(xi);
                if (plane == 0) {                                             // XY, reading S21: 2 - 3 sqrt(pi) xi erfcx(xi)
                    v = 2.0 - g * xi;
                } else {                                                      // XZ, reading S25: the second grid axis is z
                    const double xiz = ky * d_perp * 0.70710678118654752440;  //   -1 + 3 sqrt(pi) (xi_z^2 / xi) erfcx(xi)
                    v = xi > 0.0 ? -1.0 + g * (xiz * xiz / xi) : -1.0;
                }
            } else {
                const double kz = wavenumber(mz, nz, dz);
                const double k2 = kx * kx + ky * ky + kz * kz;
                if (k2 > 0.0) {                                               // readings S3, S4
                    v = 3.0 * kz * kz / k2 - 1.0;
                    if (cutoff > 0.0) {                                       // reading S5
                        const double kr = sqrt(k2) * cutoff;
                        v *= 1.0 + 3.0 * cos(kr) / (kr * kr) - 3.0 * sin(kr) / (kr * kr * kr);
                    }
                }
            }
        }
        vdd[i] = v * invP;
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return (int)e_; } while (0)

template <class K> static int set_smem(K kernel, size_t bytes) {
    if (bytes > 48 * 1024)
        CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return 0;
}

template <int N> struct PlanOf;
template <> struct PlanOf<16>  { typedef FftPlan<1, 1, true> X;  typedef FftPlan<1, 1, false> S; };
template <> struct PlanOf<32>  { typedef FftPlan<2, 1, true> X;  typedef FftPlan<2, 1, false> S; };
template <> struct PlanOf<64>  { typedef FftPlan<4, 1, true> X;  typedef FftPlan<4, 1, false> S; };
template <> struct PlanOf<128> { typedef FftPlan<8, 1, true> X;  typedef FftPlan<8, 1, false> S; };
template <> struct PlanOf<256> { typedef FftPlan<16, 1, true> X; typedef FftPlan<16, 1, false> S; };
template <> struct PlanOf<512> { typedef FftPlan<16, 2, true> X; typedef FftPlan<16, 2, false> S; };

#define DISPATCH_N(n, CALL)                                  \
    switch (n) {                                             \
        case 16:  { constexpr int N_ = 16;  CALL; } break;   \
        case 32:  { constexpr int N_ = 32;  CALL; } break;   \
        case 64:  { constexpr int N_ = 64;  CALL; } break;   \
        case 128: { constexpr int N_ = 128; CALL; } break;   \
        case 256: { constexpr int N_ = 256; CALL; } break;   \
        case 512: { constexpr int N_ = 512; CALL; } break;   \
        default: return (int)cudaErrorInvalidValue;          \
    }

static const int XTHREADS = 256;   // threads per block of k_density_fftx
static const int NLTHREADS = 128;  // threads per block of k_ifftx_nonlin

template <int N> static int launch_density_fftx(dbec_handle_s* h, int advance) {
    typedef typename PlanOf<N>::X P;
    constexpr int LP = XTHREADS / P::T;
    const int ppm = h->ny * h->nz / 2, npairs = ppm * h->nb;
    const size_t sm = (size_t)LP * XLine<P>::SMF * sizeof(cd);
    auto k = k_density_fftx<P, LP>;
    int rc = set_smem(k, sm);
    if (rc) return rc;
    cudaError_t e = launch_pdl(k, dim3((npairs + LP - 1) / LP), dim3(P::T * LP), sm, h->stream, h->use_pdl, h->psi, h->spec,
                               h->ax[0].twA, h->ax[0].twN, h->scal, npairs, h->nxhp, ppm, h->nb, advance);
    h->launches++;
    return (int)e;
}

template <int N, int MODE> static int launch_fft_strided(dbec_handle_s* h, int axis) {
    typedef typename PlanOf<N>::S P;
    constexpr int C = DBEC_SPEC_COLS;
    constexpr int TILES = (P::T * C >= 128) ? 1 : 128 / (P::T * C);
    long long line_stride, outer_stride, ntiles;
    int ntx;
    if (axis == 1) {        // y lines: for each plane (z, member), columns = kx
        line_stride = h->nxhp; outer_stride = (long long)h->ny * h->nxhp; ntx = h->nxhp / C;
        ntiles = (long long)ntx * h->nplanes;
    } else {                // z lines: columns = (ky, kx) flattened; outer = batch member
        line_stride = (long long)h->ny * h->nxhp; outer_stride = h->SP; ntx = (int)(line_stride / C);
        ntiles = (long long)ntx * h->nb;
    }
    // the multiply by V_dd rides on the last axis only: y in 2-D (table [nyf][nxhp]), z in 3-D ([nzf][nyf][nxhp])
    const int ny3 = axis == 2 ? h->ny : 0;
    const long long vls = axis == 2 ? (long long)h->nyf * h->nxhp : h->nxhp;
    const size_t sm = (size_t)TILES * P::SMEM * C * sizeof(cd);
    auto k = k_fft_strided<P, MODE, TILES>;
    int rc = set_smem(k, sm);
    if (rc) return rc;
    cudaError_t e = launch_pdl(k, dim3((unsigned)((ntiles + TILES - 1) / TILES)), dim3(P::T * C * TILES), sm, h->stream, h->use_pdl,
                               h->spec, (const double*)h->vdd, h->ax[axis].twA, h->ax[axis].twN, line_stride, outer_stride, ntx, ntiles, N, h->nxhp, ny3, vls);
    h->launches++;
    return (int)e;
}

template <int N, bool RT, int MODE> static int launch_ifftx(dbec_handle_s* h, double* phi) {
    typedef typename PlanOf<N>::X P;
    constexpr int LP = NLTHREADS / P::T;
    const int npairs = h->ny * h->nz / 2 * h->nb;
    const size_t sm = (size_t)LP * XLine<P>::SM * sizeof(cd) +
                      (MODE == NL_STEP_CNX ? 3 * cn_tab_elems(N) * sizeof(typename CnCoef<RT>::type) : 0);
    auto k = k_ifftx_nonlin<P, LP, RT, MODE>;
    int rc = set_smem(k, sm);
    if (rc) return rc;
    cudaError_t e = launch_pdl(k, dim3((npairs + LP - 1) / LP), dim3(P::T * LP), sm, h->stream, h->use_pdl,
                               (const cd*)h->spec, h->psi, phi, h->ax[0].twA, h->ax[0].twN, (const double*)h->scal, h->ax[0].vtrap,
                               h->ax[1].vtrap, h->ax[2].vtrap, h->p.dt, npairs, h->nxhp, h->ny, h->nz, make_cntab<RT>(h->ax[0]));
    h->launches++;
    return (int)e;
}

int dbec_launch_density_fftx(dbec_handle_s* h, int advance) {
    int rc;
    DISPATCH_N(h->nx, rc = launch_density_fftx<N_>(h, advance));
    return rc;
}

// mode: 0 forward, 1 inverse, 2 forward * V_dd * inverse; axis 1 (y) or 2 (z)
int dbec_launch_fft_strided(dbec_handle_s* h, int axis, int mode) {
    int rc;
    const int n = axis == 1 ? h->ny : h->nz;
    if (mode == MODE_FWD) { DISPATCH_N(n, rc = (launch_fft_strided<N_, MODE_FWD>(h, axis))); }
    else if (mode == MODE_INV) { DISPATCH_N(n, rc = (launch_fft_strided<N_, MODE_INV>(h, axis))); }
    else { DISPATCH_N(n, rc = (launch_fft_strided<N_, MODE_FMI>(h, axis))); }
    return rc;
}

int dbec_launch_nonlinear(dbec_handle_s* h, int fuse_cnx) {
    int rc;
    if (h->p.time_mode == 1) {
        if (fuse_cnx) { DISPATCH_N(h->nx, rc = (launch_ifftx<N_, true, NL_STEP_CNX>(h, nullptr))); }
        else          { DISPATCH_N(h->nx, rc = (launch_ifftx<N_, true, NL_STEP>(h, nullptr))); }
    } else {
        if (fuse_cnx) { DISPATCH_N(h->nx, rc = (launch_ifftx<N_, false, NL_STEP_CNX>(h, nullptr))); }
        else          { DISPATCH_N(h->nx, rc = (launch_ifftx<N_, false, NL_STEP>(h, nullptr))); }
    }
    return rc;
}

int dbec_launch_phi_out(dbec_handle_s* h, double* phi) {
    int rc;
    DISPATCH_N(h->nx, rc = (launch_ifftx<N_, false, NL_PHI>(h, phi)));
    return rc;
}

int dbec_launch_build_vdd(dbec_handle_s* h) {
    k_build_vdd<<<h->num_sms * 8, 256, 0, h->stream>>>(h->vdd, h->p.ndim, h->p.plane, h->nx, h->ny, h->nz, h->nxhp, h->nyf, h->nzf, h->p.dx, h->p.dy,
                                                 h->p.dz, h->p.d_perp, h->p.cutoff, 1.0 / (double)h->P);
    h->launches++;
    return (int)cudaGetLastError();
}
