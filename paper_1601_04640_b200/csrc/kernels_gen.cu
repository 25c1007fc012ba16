// kernels_gen.cu — every pass of the step for grid lines whose length is NOT one of the powers of two the
// register-resident kernels are built for: any N = 2^a 3^b 5^c 7^d, 4 <= N <= 1024 (the paper's own
// experiment sweeps 50^3 .. 600^3 and 1000^2 .. 15000^2 and advises "experimenting with different grid sizes",
// PAPER.md:81, :89, :93).  Same arithmetic as kernels_fft.cu / kernels_cn.cu (calcpsidd2, calcnu, calclux/y/z,
// calcnorm — PAPER.md:63, :67, :71, :79); what changes is that the line length is a run-time number:
//   * the line FFT is a Stockham autosort transform in shared memory, one radix-r pass (r = 4, 2, 3, 5, 7) per
//     factor of N, twiddles from the axis' table exp(-2 pi i j / N);
//   * the Crank-Nicolson solve is the chunked Thomas scheme of cn_chunk.cuh with ceil(N / 16) chunks, the last
//     one padded with h = 0 (a padded point solves to 0 and feeds nothing back).
// A handle may mix: an axis of 96 points runs here, an axis of 256 points in the persistent kernels.
#include "dbec_internal.hpp"
#include "fft_line.cuh"
#include "fft_gen.cuh"
#include "cn_chunk.cuh"
#include "cn_line_smem.cuh"
#include "tma_pipe.cuh"
#include "norm_finish.cuh"
#include "trig.cuh"

// Blocks of the FFT kernels: 256 threads, four per SM (64 registers).  Measured against 512 x 2 with the tile sizes
// below: 384^3 4.91 -> 4.57 ms per step, 320^3 2.60 -> 2.45, 192^3 0.579 -> 0.547 (more, smaller blocks overlap each
// other's load, transform and store phases; 256 x 3 with 80 registers spills less and is slower: 5.10 ms).
#define GEN_T 256
#define GEN_B 4
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return (int)e_; } while (0)

// ------------------------------------------------------------------------------------------------
// a1, x axis: n = |s psi|^2 -> half spectrum, two real lines per complex transform
// ------------------------------------------------------------------------------------------------
// Block = LP line pairs; shared memory: two buffers of LP lines of n complex values.
__global__ void __launch_bounds__(GEN_T, GEN_B)
k_gen_density_fftx(const cd* __restrict__ psi, cd* __restrict__ spec, const cd* __restrict__ twN, double* __restrict__ scal,
                   const __grid_constant__ GenPlanP pl, int LP, int npairs, int nxhp, int pairs_per_member, int nb, int advance) {
    extern __shared__ cd gsm[];
    pdl_launch_dependents(); pdl_wait();
    const int n = pl.n;
    cd* a = gsm; cd* b = gsm + (size_t)LP * n;
    const long long pair0 = (long long)blockIdx.x * LP;
    const FastDiv fn(n), fnxhp(nxhp), fone(1), fLP(LP);
    for (int idx = threadIdx.x; idx < LP * n; idx += blockDim.x) {
        int l, x;
        fn.divmod(idx, l, x);
        const long long pair = pair0 + l;
        cd v = cmake(0.0, 0.0);
        if (pair < npairs) {
            const double s2 = scal[(pair / pairs_per_member) * SC_COUNT + SC_S2];
            v = cmake(s2 * cnorm2(psi[pair * 2 * n + x]), s2 * cnorm2(psi[(pair * 2 + 1) * n + x]));
        }
        a[idx] = v;
    }
    if (advance && blockIdx.x == 0)            // first kernel of a step: move the NSTP ramp on (reads neither G nor D)
        for (int m = threadIdx.x; m < nb; m += blockDim.x) ramp_advance(scal + (size_t)m * SC_COUNT);
    __syncthreads();
    const cd* z = gen_fft_lines2<-1, false, true>(a, b, LP, fone, fLP, n, 0, 1, pl, twN);
    for (int idx = threadIdx.x; idx < LP * nxhp; idx += blockDim.x) {
        int l, k;
        fnxhp.divmod(idx, l, k);
        const long long pair = pair0 + l;
        if (pair >= npairs) continue;
        cd xa = cmake(0.0, 0.0), xb = xa;
        if (k <= n / 2) {
            const cd zk = z[l * n + k], zp = z[l * n + (k ? n - k : 0)];
            // X_a = (Z[k] + conj Z[N-k])/2,  X_b = (Z[k] - conj Z[N-k])/(2i)
            xa = cmake(0.5 * (zk.x + zp.x), 0.5 * (zk.y - zp.y));
            xb = cmake(0.5 * (zk.y + zp.y), -0.5 * (zk.x - zp.x));
        }
        spec[pair * 2 * nxhp + k] = xa;
        spec[(pair * 2 + 1) * nxhp + k] = xb;
    }
}

// ------------------------------------------------------------------------------------------------
// a1 / a3 along y or z on the half spectrum; MODE 2 = forward * V_dd(k)/P * inverse (a2 fused)
// ------------------------------------------------------------------------------------------------
// A tile is `cols` neighbouring columns (8: one 128-byte row per line point; 4 for lines longer than 256 points,
// so that four blocks with two buffers of n x cols values each fit an SM), element (j, col) at j*cols + col in
// shared memory.
template <int MODE>
__global__ void __launch_bounds__(GEN_T, GEN_B)
k_gen_fft_strided(cd* __restrict__ spec, const double* __restrict__ vdd, const cd* __restrict__ twN, const __grid_constant__ GenPlanP pl, int cols,
                  long long line_stride, long long outer_stride, int ntiles_x, long long ntiles, int nxhp, int ny3,
                  long long vdd_line_stride) {
    extern __shared__ cd gsm[];
    pdl_launch_dependents(); pdl_wait();
    const int n = pl.n;
    cd* a = gsm; cd* b = gsm + (size_t)n * cols;
    const long long tile = blockIdx.x;
    if (tile >= ntiles) return;
    const long long outer = tile / ntiles_x, tx = tile % ntiles_x;
    cd* g = spec + outer * outer_stride + tx * cols;
    const int cs = cols == 8 ? 3 : 2, cm = cols - 1;           // cols is 8 or 4
    const FastDiv fc(cols), fnxhp(nxhp);
    for (int idx = threadIdx.x; idx < n * cols; idx += blockDim.x) a[idx] = g[(long long)(idx >> cs) * line_stride + (idx & cm)];
    __syncthreads();
    cd* r = a; cd* o = b;
    if (MODE == 0 || MODE == 2) { r = gen_fft_lines2<-1, true, true>(a, b, cols, fc, fc, 1, 0, cols, pl, twN); o = (r == a) ? b : a; }
    if (MODE == 2) {
        // folded V_dd table (kernels_fft.cu: k_fft_strided): row j -> min(j, n - j); 3-D: k_y of the column folds too
        for (int idx = threadIdx.x; idx < n * cols; idx += blockDim.x) {
            const int j = idx >> cs;
            const long long cix = tx * cols + (idx & cm);
            long long voff = cix;
            if (ny3) { int ky, kx; fnxhp.divmod((int)cix, ky, kx); voff = (long long)(ky < ny3 - ky ? ky : ny3 - ky) * nxhp + kx; }
            r[idx] = cmul(vdd[voff + (long long)(j < n - j ? j : n - j) * vdd_line_stride], r[idx]);
        }
        __syncthreads();
    }
    if (MODE == 1 || MODE == 2) r = gen_fft_lines2<+1, true, true>(r, o, cols, fc, fc, 1, 0, cols, pl, twN);
    for (int idx = threadIdx.x; idx < n * cols; idx += blockDim.x) g[(long long)(idx >> cs) * line_stride + (idx & cm)] = r[idx];
}

// ------------------------------------------------------------------------------------------------
// a3 (x axis, complex-to-real, two lines per transform) + a4 calcnu, or Phi_dd written out
// ------------------------------------------------------------------------------------------------
template <bool RT, bool PHI>
__global__ void __launch_bounds__(GEN_T, GEN_B)
k_gen_ifftx_nonlin(const cd* __restrict__ spec, cd* __restrict__ psi, double* __restrict__ phi_out, const cd* __restrict__ twN,
                   const double* __restrict__ scal, const double* __restrict__ vx, const double* __restrict__ vy,
                   const double* __restrict__ vz, double dt, const __grid_constant__ GenPlanP pl, int LP, int npairs, int nxhp, int ny, int nz) {
    extern __shared__ cd gsm[];
    pdl_launch_dependents(); pdl_wait();
    const int n = pl.n;
    cd* a = gsm; cd* b = gsm + (size_t)LP * n;
    const long long pair0 = (long long)blockIdx.x * LP;
    const FastDiv fn(n), fone(1), fLP(LP);
    for (int idx = threadIdx.x; idx < LP * n; idx += blockDim.x) {
        int l, k;
        fn.divmod(idx, l, k);
        const long long pair = pair0 + l;
        cd v = cmake(0.0, 0.0);
        if (pair < npairs) {
            const cd* sa = spec + pair * 2 * nxhp;
            const cd* sb = sa + nxhp;
            if (k <= n / 2) { const cd p = sa[k], q = sb[k]; v = cmake(p.x - q.y, p.y + q.x); }            // X_a + i X_b
            else { const cd p = sa[n - k], q = sb[n - k]; v = cmake(p.x + q.y, q.x - p.y); }               // conj X_a + i conj X_b
        }
        a[idx] = v;
    }
    __syncthreads();
    const cd* f = gen_fft_lines2<+1, false, true>(a, b, LP, fone, fLP, n, 0, 1, pl, twN);      // (Phi on line a, Phi on line b); 1/P is in the table
    for (int idx = threadIdx.x; idx < 2 * LP * n; idx += blockDim.x) {
        int ll, x;
        fn.divmod(idx, ll, x);                              // line ll of the block: pair ll / 2, component ll & 1
        const long long row = (pair0 + ll / 2) * 2 + (ll & 1);
        if (row >= 2LL * npairs) continue;
        const cd pp = f[(ll / 2) * n + x];
        const double phi = (ll & 1) ? pp.y : pp.x;
        if (PHI) { phi_out[row * n + x] = phi; continue; }
        const int y = (int)(row % ny), zz = (int)(row / ny), z = zz % nz;
        const double* sc = scal + (size_t)(zz / nz) * SC_COUNT;           // this row's batch member
        const double s = sc[SC_S], s2 = sc[SC_S2];
        const cd q = psi[row * n + x];
        const double u = dt * (vx[x] + vy[y] + vz[z] + sc[SC_G] * (s2 * cnorm2(q)) + sc[SC_D] * phi);
        cd r;
        if (RT) { double sn, cs; sincos_cw(u, &sn, &cs); r = cmul(s, cmul(q, cmake(cs, -sn))); }      // (trig.cuh: branch-free)
        else r = cmul(s * exp_cw(-u), q);
        psi[row * n + x] = r;
    }
}

// ------------------------------------------------------------------------------------------------
// a5..a7 (+ a8): Crank-Nicolson sweep along any axis, ceil(n / 16) chunks per line
// ------------------------------------------------------------------------------------------------
// Thread (chunk c, column col) of a tile of GC columns; point j of column q sits at q*col_stride + j*elem_stride
// (x sweep: columns are lines, elem_stride 1; y / z sweeps: columns are neighbouring x, elem_stride = line stride).
// blockIdx.y = outer index (plane or batch member).  Points j >= n of the last chunk are padding: psi = 0, h = 0.
// L: points per chunk — 8 (tables pf8 / pb8: 32 registers of psi per thread, up to 1024 threads per tile) for every
// axis; 16 stays available for comparison.
constexpr int GC = 8;
// REGS: register cap (L = 8: 64, or 56 where that lets one more block of the tile's size onto the SM)
template <bool RT, bool NORM, int L, int REGS>
__global__ void __launch_bounds__(L == 8 ? 1024 : 512) __maxnreg__(REGS)
k_gen_cn(cd* __restrict__ psi, CnTab<RT> cn, int n, int nch, long long elem_stride, long long col_stride, long long outer_stride,
         long long ncols, double* __restrict__ partial, unsigned int* ticket, double* __restrict__ scal, double dV, int nb, int K) {
    typedef typename CnCoef<RT>::type CT;
    extern __shared__ cd gsm[];                // [2][chunk slots][GC] zero-start chunk ends
    // (the block is rounded up to whole warps: chunk slots c >= nch hold padding only and solve to zero)
    const int nslot = blockDim.x / GC;
    __shared__ double red[32];
    pdl_launch_dependents(); pdl_wait();
    const int col = threadIdx.x % GC, c = threadIdx.x / GC, j0 = c * L;
    long long q = (long long)blockIdx.x * GC + col;
    const bool active = q < ncols;
    if (!active) q = 0;
    cd* g = psi + (long long)blockIdx.y * outer_stride + q * col_stride;
    const cd zero = cmake(0.0, 0.0);
    cd u[L];
#pragma unroll
    for (int i = 0; i < L; ++i) u[i] = (j0 + i < n) ? g[(j0 + i) * elem_stride] : zero;
    // the tables are zero-padded to whole chunks (dbec_api.cu: upload_axis); chunk slots beyond them read chunk 0
    const int jt = j0 < n ? j0 : 0;
    const bool pad = j0 >= n;
    const cd lo = (j0 > 0 && j0 - 1 < n) ? g[(j0 - 1) * elem_stride] : zero;
    const cd hi = (j0 + L < n) ? g[(j0 + L) * elem_stride] : zero;
    cn_chunk_forward<CT>(u, lo, hi, cn.kap, cn.h + jt);
    if (pad) {
#pragma unroll
        for (int i = 0; i < L; ++i) u[i] = zero;
    }
    cd* e0 = gsm; cd* e1 = gsm + nslot * GC;
    e0[c * GC + col] = u[L - 1];
    __syncthreads();
    // carries over ALL earlier / later chunks; chunk-end products from the per-element tables
    cd din = zero;
    // (the carry is a Horner sum over the earlier chunk ends with factors < 1: the host counts the K terms that are
    // above 2^-73 of the first, dbec_api.cu carry_terms; the rest is below the last bit of the sum)
    for (int i = (c - K > 0 ? c - K : 0); i < c && i < nch; ++i) din = cn_fma(cn.pf[i * L + L - 1], din, e0[i * GC + col]);
    cn_chunk_backward<CT>(u, din, cn.h + jt, cn.pf + jt);
    if (pad) {
#pragma unroll
        for (int i = 0; i < L; ++i) u[i] = zero;
    }
    e1[c * GC + col] = u[0];
    __syncthreads();
    cd uin = zero;
    for (int i = (c + K < nch - 1 ? c + K : nch - 1); i > c; --i) uin = cn_fma(cn.pb[i * L], uin, e1[i * GC + col]);
    cn_chunk_fix<CT>(u, uin, cn.pb + jt);
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < L; ++i) {
        if (active && j0 + i < n) { g[(j0 + i) * elem_stride] = u[i]; if (NORM) acc += cnorm2(u[i]); }
    }
    if (NORM) {
        // block sum in a fixed order, then the last block's per-member finish (kernels_cn.cu)
        double x = acc;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
        __syncthreads();
        if (l == 0) red[w] = x;
        __syncthreads();
        double part = 0.0;
        if (threadIdx.x == 0) for (int i = 0; i < nw; ++i) part += red[i];
        __syncthreads();
        norm_finish(part, partial, ticket, scal, dV, red, nb);
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
// Radices of a length with factors 2, 3, 5, 7 only: 4s first, then one 2, then the odd ones.  Returns the number
// of radices, 0 if n has another prime factor.
int dbec_gen_factor(int n, int* fac) {
    int k = 0;
    while (n % 4 == 0) { fac[k++] = 4; n /= 4; }
    if (n % 2 == 0) { fac[k++] = 2; n /= 2; }
    for (int p = 3; p <= 7; p += 2) while (n % p == 0) { fac[k++] = p; n /= p; }
    return n == 1 ? k : 0;
}

// The plans of this file take the powers of two in passes of radix 16 and 8 first (384 = 16 x 8 x 3: three passes
// through shared memory instead of five).
static GenPlanP plan_of(const dbec_handle_s* h, int axis) {
    GenPlan pl;
    int n = h->ax[axis].n, k = 0;
    pl.n = n;
    for (int i = 0; i < 12; ++i) pl.fac[i] = 0;
    while (n % 8 == 0) { pl.fac[k++] = 8; n /= 8; }
    k += dbec_gen_factor(n, pl.fac + k);
    pl.nfac = k;
    GenPlanP pp;
    make_plan_p(pl, &pp);
    return pp;
}

template <class K> static int gen_smem(K kernel, size_t bytes) {
    if (bytes > 48 * 1024) CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return 0;
}

// line pairs per block of the x kernels: two buffers of LP lines within 48 KiB (four blocks per SM)
static int gen_lp(int n) { int lp = 1536 / n; return lp < 1 ? 1 : (lp > 8 ? 8 : lp); }

int dbec_launch_gen_density_fftx(dbec_handle_s* h, int advance) {
    const GenPlanP pl = plan_of(h, 0);
    const int LP = gen_lp(pl.n), ppm = h->ny * h->nz / 2, npairs = ppm * h->nb;
    const size_t sm = 2 * (size_t)LP * pl.n * sizeof(cd);
    CK((cudaError_t)gen_smem(k_gen_density_fftx, sm));
    CK(launch_pdl(k_gen_density_fftx, dim3((npairs + LP - 1) / LP), dim3(GEN_T), sm, h->stream, h->use_pdl, (const cd*)h->psi, h->spec,
                  h->ax[0].twN, h->scal, pl, LP, npairs, h->nxhp, ppm, h->nb, advance));
    h->launches++;
    return (int)cudaGetLastError();
}

template <int MODE> static int launch_gen_fft(dbec_handle_s* h, int axis) {
    const GenPlanP pl = plan_of(h, axis);
    const int cols = pl.n <= 256 ? 8 : 4;          // two buffers of n x cols values within 48 KiB up to n = 384
    long long line_stride, outer_stride, ntiles;
    int ntx;
    if (axis == 1) { line_stride = h->nxhp; outer_stride = (long long)h->ny * h->nxhp; ntx = h->nxhp / cols; ntiles = (long long)ntx * h->nplanes; }
    else { line_stride = (long long)h->ny * h->nxhp; outer_stride = h->SP; ntx = (int)(line_stride / cols); ntiles = (long long)ntx * h->nb; }
    const int ny3 = axis == 2 ? h->ny : 0;
    const long long vls = axis == 2 ? (long long)h->nyf * h->nxhp : h->nxhp;
    const size_t sm = 2 * (size_t)pl.n * cols * sizeof(cd);
    auto k = k_gen_fft_strided<MODE>;
    CK((cudaError_t)gen_smem(k, sm));
    CK(launch_pdl(k, dim3((unsigned)ntiles), dim3(GEN_T), sm, h->stream, h->use_pdl, h->spec, (const double*)h->vdd, h->ax[axis].twN, pl,
                  cols, line_stride, outer_stride, ntx, ntiles, h->nxhp, ny3, vls));
    h->launches++;
    return (int)cudaGetLastError();
}

int dbec_launch_gen_fft(dbec_handle_s* h, int axis, int mode) {
    return mode == 0 ? launch_gen_fft<0>(h, axis) : mode == 1 ? launch_gen_fft<1>(h, axis) : launch_gen_fft<2>(h, axis);
}

template <bool RT, bool PHI> static int launch_gen_nonlin(dbec_handle_s* h, double* phi) {
    const GenPlanP pl = plan_of(h, 0);
    const int LP = gen_lp(pl.n), npairs = h->ny * h->nz / 2 * h->nb;
    const size_t sm = 2 * (size_t)LP * pl.n * sizeof(cd);
    auto k = k_gen_ifftx_nonlin<RT, PHI>;
    CK((cudaError_t)gen_smem(k, sm));
    CK(launch_pdl(k, dim3((npairs + LP - 1) / LP), dim3(GEN_T), sm, h->stream, h->use_pdl, (const cd*)h->spec, h->psi, phi, h->ax[0].twN,
                  (const double*)h->scal, h->ax[0].vtrap, h->ax[1].vtrap, h->ax[2].vtrap, h->p.dt, pl, LP, npairs, h->nxhp, h->ny, h->nz));
    h->launches++;
    return (int)cudaGetLastError();
}

int dbec_launch_gen_nonlinear(dbec_handle_s* h) {
    return h->p.time_mode == 1 ? launch_gen_nonlin<true, false>(h, nullptr) : launch_gen_nonlin<false, false>(h, nullptr);
}
int dbec_launch_gen_phi_out(dbec_handle_s* h, double* phi) { return launch_gen_nonlin<false, true>(h, phi); }

// chunk tables of 8 points as a CnTab (cn_line_smem.cuh holds the 16-point ones)
template <bool RT> static CnTab<RT> cntab8(const AxisTables& a);
template <> CnTab<true> cntab8<true>(const AxisTables& a) {
    CnTab<true> t; t.h = a.h; t.pf = a.pf8; t.pb = a.pb8; t.pfe = a.pfe8; t.pbs = a.pbs8; t.kap = a.kap; t.K = a.K8; return t;
}
template <> CnTab<false> cntab8<false>(const AxisTables& a) {
    CnTab<false> t; t.h = a.h_re; t.pf = a.pf8_re; t.pb = a.pb8_re; t.pfe = a.pfe8_re; t.pbs = a.pbs8_re; t.kap = a.kap.x; t.K = a.K8;
    return t;
}

// Chunks of 8 points along y and z (measured at 384^3 and 320^3: 5 - 20 % faster than 16), of 16 along x, where a
// thread's chunk is contiguous in memory and 8-point chunks leave half of every 256 bytes to another warp.
template <bool RT, bool NORM, int L, int REGS> static int launch_gen_cn_l(dbec_handle_s* h, int axis) {
    const int n = h->ax[axis].n, nch = (n + L - 1) / L;
    const int threads = (nch * GC + 31) / 32 * 32;
    long long es, cs, os, ncols;
    int nouter;
    if (axis == 0) { es = 1; cs = h->nx; os = 0; ncols = (long long)h->ny * h->nplanes; nouter = 1; }
    else if (axis == 1) { es = h->nx; cs = 1; os = (long long)h->nx * h->ny; ncols = h->nx; nouter = h->nplanes; }
    else { es = (long long)h->nx * h->ny; cs = 1; os = h->P; ncols = es; nouter = h->nb; }
    dim3 grid((unsigned)((ncols + GC - 1) / GC), (unsigned)nouter);
    if (NORM && (long long)grid.x * grid.y > h->npartial) return (int)cudaErrorInvalidValue;
    const size_t sm = 2 * (size_t)(threads / GC) * GC * sizeof(cd);
    CK(launch_pdl(k_gen_cn<RT, NORM, L, REGS>, grid, dim3(threads), sm, h->stream, h->use_pdl, h->psi,
                  L == 8 ? cntab8<RT>(h->ax[axis]) : make_cntab<RT>(h->ax[axis]), n, nch, es, cs, os,
                  ncols, h->partial, h->ticket, h->scal, h->dV, h->nb, L == 8 ? h->ax[axis].K8 : h->ax[axis].K16));
    h->launches++;
    return (int)cudaGetLastError();
}

template <bool RT, bool NORM> static int launch_gen_cn(dbec_handle_s* h, int axis) {
    if (axis == 0) return launch_gen_cn_l<RT, NORM, 16, 128>(h, axis);
    // 8-point chunks: 64 registers hold a chunk without spilling much; 56 cost a few more spills and pay when they
    // let one more block onto the SM (measured at 384^3: 384 threads per block, 2 -> 3 blocks, sweeps 515 -> 447 us;
    // at 320^3, 3 blocks either way, 258 -> 284 us)
    const int threads = ((h->ax[axis].n + 7) / 8 * GC + 31) / 32 * 32;
    const bool r56 = 65536 / (threads * 56) > 65536 / (threads * 64);
    return r56 ? launch_gen_cn_l<RT, NORM, 8, 56>(h, axis) : launch_gen_cn_l<RT, NORM, 8, 64>(h, axis);
}

int dbec_launch_gen_cn(dbec_handle_s* h, int axis, int with_norm) {
    if (axis == 0 && with_norm) return (int)cudaErrorInvalidValue;
    if (h->p.time_mode == 1) return with_norm ? launch_gen_cn<true, true>(h, axis) : launch_gen_cn<true, false>(h, axis);
    return with_norm ? launch_gen_cn<false, true>(h, axis) : launch_gen_cn<false, false>(h, axis);
}
