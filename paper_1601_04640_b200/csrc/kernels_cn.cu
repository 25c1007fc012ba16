// kernels_cn.cu — Crank-Nicolson sweeps (calclux / calcluy / calcluz), the norm
// (calcnorm) and the observables (calcmuen, calcrms).
//
// The paper gives each grid line to one thread that runs the whole "recursive relation" and keeps
// its coefficient array in global memory.  Here a line is cut into chunks of 16 points
// held in registers, one thread per chunk, and the chunks are tied together by an exact carry
// recurrence over the chunk ends (cn_chunk.cuh), so a tile of lines is read once and written once:
//   k_cn_strided   y or z sweep: a tile of COLS neighbouring lines; every global access is a run of
//                  COLS consecutive complex128 values (COLS x 16 B).  Optionally accumulates the
//                  block's sum of |psi|^2 and lets the last block turn the partial sums into the
//                  deferred norm factor (imaginary time), so that calcnorm costs no pass of its own.
//   k_cn_x         x sweep alone: lines are contiguous; coalesced loads, transposition through a
//                  padded shared row (cn_line_smem.cuh).
#include "dbec_internal.hpp"
#include "cn_chunk.cuh"
#include "cn_line_smem.cuh"
#include "tma_pipe.cuh"
#include "norm_finish.cuh"

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return (int)e_; } while (0)

// Sum over the block in a fixed order (warp shuffles, then warp 0 over the warp sums).
template <int NT> __device__ __forceinline__ double block_sum(double x, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    constexpr int NW = (NT + 31) / 32;
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) red[w] = x;
    __syncthreads();
    double t = (threadIdx.x < NW) ? red[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;   // valid in thread 0
}

__device__ __forceinline__ double block_max(double x, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_down_sync(0xffffffffu, x, o));
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (l == 0) red[w] = x;
    __syncthreads();
    double t = (threadIdx.x < nw) ? red[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t = fmax(t, __shfl_down_sync(0xffffffffu, t, o));
    }
    return t;
}

// ------------------------------------------------------------------------------------------------
// strided sweeps
// ------------------------------------------------------------------------------------------------
template <bool RT, int NCH, int COLS, bool NORM>
__global__ void __launch_bounds__(NCH* COLS, (NCH * COLS <= 256 ? 2 : 1))
k_cn_strided(cd* __restrict__ psi, CnTab<RT> cn, long long line_stride, long long outer_stride, long long ncols,
             double* __restrict__ partial, unsigned int* ticket, double* __restrict__ scal, double dV, int nb) {
    typedef typename CnCoef<RT>::type CT;
    __shared__ cd edge[2][NCH][COLS];     // first and last point of every chunk (halo of the neighbours)
    __shared__ cd ends[2][NCH][COLS];     // zero-start chunk results for the carries
    __shared__ double red[32];
    pdl_launch_dependents(); pdl_wait();       // (tma_pipe.cuh) launch latency overlaps the previous kernel
    const int col = threadIdx.x % COLS, c = threadIdx.x / COLS;
    long long gcol = (long long)blockIdx.x * COLS + col;
    const bool active = gcol < ncols;          // narrow grids: a tile may be wider than the grid
    if (!active) gcol = 0;
    cd* g = psi + (long long)blockIdx.y * outer_stride + gcol + (long long)(c * CN_L) * line_stride;
    cd u[CN_L];
#pragma unroll
    for (int i = 0; i < CN_L; ++i) u[i] = g[i * line_stride];
    if (NCH > 1) {
        edge[0][c][col] = u[0];
        edge[1][c][col] = u[CN_L - 1];
        __syncthreads();
    }
    const cd lo = (c > 0) ? edge[1][c - 1][col] : cmake(0.0, 0.0);
    const cd hi = (c < NCH - 1) ? edge[0][c + 1][col] : cmake(0.0, 0.0);
    const int j0 = c * CN_L;
    cn_chunk_forward<CT>(u, lo, hi, cn.kap, cn.h + j0);
    cd din = cmake(0.0, 0.0), uin = cmake(0.0, 0.0);
    if (NCH > 1) {
        ends[0][c][col] = u[CN_L - 1];
        __syncthreads();
        din = cn_carry_forward<CT>(c, &ends[0][0][col], COLS, cn.pfe);
    }
    cn_chunk_backward<CT>(u, din, cn.h + j0, cn.pf + j0);
    if (NCH > 1) {
        ends[1][c][col] = u[0];
        __syncthreads();
        uin = cn_carry_backward<CT>(c, NCH, &ends[1][0][col], COLS, cn.pbs);
    }
    cn_chunk_fix<CT>(u, uin, cn.pb + j0);
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < CN_L; ++i) {
        if (active) {
            g[i * line_stride] = u[i];
            if (NORM) acc += cnorm2(u[i]);
        }
    }
    if (NORM) {
        const double part = block_sum<NCH * COLS>(acc, red);
        norm_finish(part, partial, ticket, scal, dV, red, nb);
    }
}

// ------------------------------------------------------------------------------------------------
// x sweep alone
// ------------------------------------------------------------------------------------------------
template <bool RT, int T, int LPB>
__global__ void __launch_bounds__(T* LPB)
k_cn_x(cd* __restrict__ psi, CnTab<RT> cn, int nlines) {
    extern __shared__ cd smem[];
    typedef typename CnCoef<RT>::type CT;
    pdl_launch_dependents(); pdl_wait();
    constexpr int N = 16 * T;
    const int lp = threadIdx.x / T, m = threadIdx.x % T;
    long long line = (long long)blockIdx.x * LPB + lp;
    const bool active = line < nlines;
    if (!active) line = 0;
    const CnTab<RT> cs = cn_stage_tables<RT, N>(cn, (CT*)smem);
    cd* sm = smem + (3 * cn_tab_elems(N) * sizeof(CT)) / sizeof(cd) + lp * (N + 3 * T);
    cd* g = psi + line * N;
    cd q[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) q[j] = g[j * T + m];
    __syncthreads();
    cn_line_via_smem<RT, T, 17>(q, m, sm, cs);
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        if (active) g[j * T + m] = q[j];
    }
}

// ------------------------------------------------------------------------------------------------
// calcnorm alone, psi <- s psi, and the observables
// ------------------------------------------------------------------------------------------------
// grid (blocks per member, members): blockIdx.y is the batch member
__global__ void __launch_bounds__(256)
k_norm(const cd* __restrict__ psi, long long P, double* __restrict__ partial, unsigned int* ticket,
       double* __restrict__ scal, double dV) {
    __shared__ double red[32];
    const cd* p = psi + (size_t)blockIdx.y * P;
    double acc = 0.0;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < P; i += (long long)gridDim.x * 256)
        acc += cnorm2(p[i]);
    const double part = block_sum<256>(acc, red);
    norm_finish(part, partial, ticket, scal, dV, red, gridDim.y);
}

__global__ void __launch_bounds__(256) k_apply_scale(cd* __restrict__ psi, long long P, const double* __restrict__ scal) {
    const double s = scal[(size_t)blockIdx.y * SC_COUNT + SC_S];
    cd* p = psi + (size_t)blockIdx.y * P;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < P; i += (long long)gridDim.x * 256)
        p[i] = cmul(s, p[i]);
}
__global__ void k_reset_scale(double* scal, int nb) {
    for (int b = threadIdx.x; b < nb; b += blockDim.x) { scal[(size_t)b * SC_COUNT + SC_S] = 1.0; scal[(size_t)b * SC_COUNT + SC_S2] = 1.0; }
}

// Observable partial sums (reading S13, S14; definitions in DESIGN.md "Observables"), per block:
//   0 sum n   1 sum x^2 n   2 sum y^2 n   3 sum z^2 n   4 sum n^2   5 sum Phi n
//   6 sum |psi(x+1)-psi|^2   7 same along y   8 same along z   9 max n
enum { OB_N = 0, OB_X2, OB_Y2, OB_Z2, OB_N2, OB_PHIN, OB_KX, OB_KY, OB_KZ, OB_MAX, OB_COUNT };

// grid (blocks per member, members).  A block walks whole x-lines (TPR threads per line, 256 / TPR lines at
// a time), so that the indices (iy, iz) cost one division per line instead of two 64-bit ones per point.
__global__ void __launch_bounds__(256)
k_obs_partial(const cd* __restrict__ psi_all, const double* __restrict__ phi_all, const double* __restrict__ scal_all,
              const double* __restrict__ x2, const double* __restrict__ y2, const double* __restrict__ z2,
              int nx, int ny, int nz, int tpr, double* __restrict__ partial_all) {
    __shared__ double red[32];
    const long long P = (long long)nx * ny * nz;
    const cd* psi = psi_all + (size_t)blockIdx.y * P;
    const double* phi = phi_all + (size_t)blockIdx.y * P;
    double* partial = partial_all + (size_t)blockIdx.y * OB_COUNT * gridDim.x;
    const double s2 = scal_all[(size_t)blockIdx.y * SC_COUNT + SC_S2];
    double a[OB_COUNT];
#pragma unroll
    for (int k = 0; k < OB_COUNT; ++k) a[k] = 0.0;
    const int lpb = 256 / tpr, lane = threadIdx.x % tpr, sub = threadIdx.x / tpr;
    const int nlines = ny * nz;
    for (int line = blockIdx.x * lpb + sub; line < nlines; line += gridDim.x * lpb) {
        const int iy = line % ny, iz = line / ny;
        const double yy = y2[iy], zz = z2[iz];
        const long long base = (long long)line * nx;
        const bool hy = iy + 1 < ny, hz = iz + 1 < nz;
        for (int ix = lane; ix < nx; ix += tpr) {
            const long long i = base + ix;
            const cd p = psi[i];
            const double n = s2 * cnorm2(p);
            a[OB_N] += n;
            a[OB_X2] += x2[ix] * n;
            a[OB_Y2] += yy * n;
            a[OB_Z2] += zz * n;
            a[OB_N2] += n * n;
            a[OB_PHIN] += phi[i] * n;
            if (ix + 1 < nx) a[OB_KX] += s2 * cnorm2(csub(psi[i + 1], p));
            if (hy) a[OB_KY] += s2 * cnorm2(csub(psi[i + nx], p));
            if (hz) a[OB_KZ] += s2 * cnorm2(csub(psi[i + (long long)nx * ny], p));
            a[OB_MAX] = fmax(a[OB_MAX], n);
        }
    }
#pragma unroll
    for (int k = 0; k < OB_COUNT; ++k) {
        const double t = (k == OB_MAX) ? block_max(a[k], red) : block_sum<256>(a[k], red);
        if (threadIdx.x == 0) partial[(long long)k * gridDim.x + blockIdx.x] = t;
    }
}

// One block: fixed-order sums over the block partials, then the observables.
__global__ void __launch_bounds__(256)
k_obs_final(const double* __restrict__ partial_all, int nb, const cd* __restrict__ psi_all, const double* __restrict__ scal_all,
            long long P, long long centre, double dV, double dx, double dy, double dz, int ndim, double nu, double lam,
            double kap, double* __restrict__ out_all) {
    __shared__ double red[32];
    __shared__ double tot[OB_COUNT];
    // one block per batch member
    const double* partial = partial_all + (size_t)blockIdx.x * OB_COUNT * nb;
    const cd* psi = psi_all + (size_t)blockIdx.x * P;
    const double* scal = scal_all + (size_t)blockIdx.x * SC_COUNT;
    double* out = out_all + (size_t)blockIdx.x * 16;
    for (int k = 0; k < OB_COUNT; ++k) {
        double acc = 0.0;
        for (int i = threadIdx.x; i < nb; i += 256)
            acc = (k == OB_MAX) ? fmax(acc, partial[(long long)k * nb + i]) : acc + partial[(long long)k * nb + i];
        const double t = (k == OB_MAX) ? block_max(acc, red) : block_sum<256>(acc, red);
        if (threadIdx.x == 0) tot[k] = t;
        __syncthreads();
    }
    if (threadIdx.x != 0) return;
    const double G = scal[SC_G], D = scal[SC_D], s2 = scal[SC_S2];
    const double S = dV * tot[OB_N];
    const double sx2 = dV * tot[OB_X2], sy2 = dV * tot[OB_Y2], sz2 = (ndim == 3) ? dV * tot[OB_Z2] : 0.0;
    const double ekin = 0.5 * dV * (tot[OB_KX] / (dx * dx) + tot[OB_KY] / (dy * dy) +
                                    (ndim == 3 ? tot[OB_KZ] / (dz * dz) : 0.0));
    const double etr = 0.5 * (nu * nu * sx2 + lam * lam * sy2 + kap * kap * sz2);
    const double ec = G * dV * tot[OB_N2];
    const double ed = D * dV * tot[OB_PHIN];
    out[0] = S;
    out[1] = (ekin + etr + ec + ed) / S;
    out[2] = (ekin + etr + 0.5 * ec + 0.5 * ed) / S;
    out[3] = sqrt(sx2 / S);
    out[4] = sqrt(sy2 / S);
    out[5] = sqrt(sz2 / S);
    out[6] = sqrt((sx2 + sy2 + sz2) / S);
    out[7] = s2 * cnorm2(psi[centre]);
    out[8] = tot[OB_MAX];
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
template <bool RT, int NCH, bool NORM> static int launch_cn_strided(dbec_handle_s* h, int axis) {
    constexpr int COLS = (NCH >= 16) ? 16 : (NCH >= 4 ? 32 : 64);      // 256 / 128 / 64..128 threads
    long long line_stride, outer_stride, ncols;
    int nouter;
    // y sweep: one block row per xy plane (planes of all members back to back); z sweep: one per member
    if (axis == 1) { line_stride = h->nx; outer_stride = (long long)h->nx * h->ny; ncols = h->nx; nouter = h->nplanes; }
    else { line_stride = (long long)h->nx * h->ny; outer_stride = h->P; ncols = line_stride; nouter = h->nb; }
    dim3 grid((unsigned)((ncols + COLS - 1) / COLS), (unsigned)nouter);
    if (NORM && (long long)grid.x * grid.y > h->npartial) return (int)cudaErrorInvalidValue;
    cudaError_t e = launch_pdl(k_cn_strided<RT, NCH, COLS, NORM>, grid, dim3(NCH * COLS), 0, h->stream, h->use_pdl, h->psi,
                               make_cntab<RT>(h->ax[axis]), line_stride, outer_stride, ncols, h->partial, h->ticket, h->scal, h->dV, h->nb);
    h->launches++;
    return (int)e;
}

template <bool RT, int NCH> static int launch_cn_x(dbec_handle_s* h) {
    constexpr int T = NCH, LPB = 256 / T;
    const int nlines = h->ny * h->nplanes;
    const size_t sm = (size_t)LPB * (16 * T + 3 * T) * sizeof(cd) +
                      3 * cn_tab_elems(16 * T) * sizeof(typename CnCoef<RT>::type);
    auto k = k_cn_x<RT, T, LPB>;
    if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const int nblk = (nlines + LPB - 1) / LPB;
    cudaError_t e = launch_pdl(k, dim3(nblk), dim3(T * LPB), sm, h->stream, h->use_pdl, h->psi, make_cntab<RT>(h->ax[0]), nlines);
    h->launches++;
    return (int)e;
}

template <bool RT, bool NORM> static int launch_cn_rt(dbec_handle_s* h, int axis) {
    const int n = h->ax[axis].n;
    if (axis == 0 && NORM) return (int)cudaErrorInvalidValue;      // the x sweep is never the last one of a step
#define CASE_(nch) case nch * 16: return axis == 0 ? launch_cn_x<RT, nch>(h) : launch_cn_strided<RT, nch, NORM>(h, axis)
    switch (n) {
        CASE_(1); CASE_(2); CASE_(4); CASE_(8); CASE_(16); CASE_(32);
        default: return (int)cudaErrorInvalidValue;
    }
#undef CASE_
}

int dbec_launch_cn(dbec_handle_s* h, int axis, int with_norm) {
    if (h->p.time_mode == 1) return with_norm ? launch_cn_rt<true, true>(h, axis) : launch_cn_rt<true, false>(h, axis);
    return with_norm ? launch_cn_rt<false, true>(h, axis) : launch_cn_rt<false, false>(h, axis);
}

int dbec_launch_normalize(dbec_handle_s* h) {
    // true psi = s * stored psi: bring the stored field to s = 1 first, then take the norm factor
    int rc = dbec_launch_apply_scale(h);
    if (rc) return rc;
    return dbec_launch_norm_only(h);
}

// Blocks per member of the member-wise reductions: enough to fill the GPU, within the partial-sum buffer.
static int blocks_per_member(const dbec_handle_s* h, int per_block_slots) {
    int n = (h->num_sms * 8 + h->nb - 1) / h->nb;
    const long long cap = (long long)h->npartial / ((long long)per_block_slots * h->nb);
    if (n > cap) n = (int)cap;
    const long long need = (h->P + 255) / 256;
    if (n > need) n = (int)need;
    return n < 1 ? 1 : n;
}

// calcnorm on the stored field (s must be 1): writes every member's factor
int dbec_launch_norm_only(dbec_handle_s* h) {
    k_norm<<<dim3(blocks_per_member(h, 1), h->nb), 256, 0, h->stream>>>(h->psi, h->P, h->partial, h->ticket, h->scal, h->dV);
    h->launches++;
    return (int)cudaGetLastError();
}

int dbec_launch_apply_scale(dbec_handle_s* h) {
    k_apply_scale<<<dim3(blocks_per_member(h, 1), h->nb), 256, 0, h->stream>>>(h->psi, h->P, h->scal);
    k_reset_scale<<<1, 128, 0, h->stream>>>(h->scal, h->nb);
    h->launches += 2;
    return (int)cudaGetLastError();
}

int dbec_launch_reset_scale(dbec_handle_s* h) {
    k_reset_scale<<<1, 128, 0, h->stream>>>(h->scal, h->nb);
    h->launches++;
    return (int)cudaGetLastError();
}

int dbec_launch_observables(dbec_handle_s* h) {
    const int nblk = blocks_per_member(h, OB_COUNT);
    int tpr = 256;
    while (tpr > h->nx) tpr >>= 1;               // threads per x-line: the largest power of two <= min(nx, 256)
    k_obs_partial<<<dim3(nblk, h->nb), 256, 0, h->stream>>>(h->psi, h->phi, h->scal, h->ax[0].x2, h->ax[1].x2, h->ax[2].x2, h->nx,
                                                            h->ny, h->nz, tpr, h->partial);
    const long long centre = (h->nx / 2) + (long long)h->nx * ((h->ny / 2) + (long long)h->ny * (h->p.ndim == 3 ? h->nz / 2 : 0));
    k_obs_final<<<h->nb, 256, 0, h->stream>>>(h->partial, nblk, h->psi, h->scal, h->P, centre, h->dV, h->p.dx, h->p.dy, h->p.dz,
                                              h->p.ndim, h->p.nu, h->p.lambda, h->p.kappa, h->obs_dev);
    h->launches += 2;
    return (int)cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// integrated densities (reading S27; the lineage's 1-D / 2-D density output)
// ------------------------------------------------------------------------------------------------
// out[j] = w * sum_{i < n} s2 |psi[base(j) + i*stride]|^2 over an index set j = (j0, j1):
// base(j) = j0*s0 + j1*s1, j0 < n0 (fastest in out), j1 < n1.  One thread per output, fixed order.
__global__ void __launch_bounds__(256)
k_density_sum(const cd* __restrict__ psi, const double* __restrict__ scal, double* __restrict__ out, int n, long long stride,
              int n0, long long s0, int n1, long long s1, double w) {
    const double s2 = scal[SC_S2] * w;
    const long long tot = (long long)n0 * n1;
    for (long long j = (long long)blockIdx.x * 256 + threadIdx.x; j < tot; j += (long long)gridDim.x * 256) {
        const cd* p = psi + (j % n0) * s0 + (j / n0) * s1;
        double a = 0.0;
        for (int i = 0; i < n; ++i) a += cnorm2(p[(long long)i * stride]);
        out[j] = s2 * a;
    }
}
// out[j] = w * sum_{i < n} in[j*s0 + i*stride]
__global__ void __launch_bounds__(256)
k_reduce_rows(const double* __restrict__ in, double* __restrict__ out, int n, long long stride, int n0, long long s0, double w) {
    for (int j = blockIdx.x * 256 + threadIdx.x; j < n0; j += gridDim.x * 256) {
        double a = 0.0;
        for (int i = 0; i < n; ++i) a += in[(long long)j * s0 + (long long)i * stride];
        out[j] = w * a;
    }
}

// 2-D density of a 3-D grid, integrated over `axis`; out: the lower remaining axis fastest.
int dbec_launch_density_2d(dbec_handle_s* h, int member, int axis, double* out) {
    const long long sx = 1, sy = h->nx, sz = (long long)h->nx * h->ny;
    const int n[3] = {h->nx, h->ny, h->nz};
    const long long st[3] = {sx, sy, sz};
    const double d[3] = {h->p.dx, h->p.dy, h->p.dz};
    const int lo = axis == 0 ? 1 : 0, hi = axis == 2 ? 1 : 2;
    const long long tot = (long long)n[lo] * n[hi];
    int nblk = (int)((tot + 255) / 256);
    if (nblk > h->num_sms * 8) nblk = h->num_sms * 8;
    k_density_sum<<<nblk, 256, 0, h->stream>>>(h->psi + (size_t)member * h->P, h->scal + (size_t)member * SC_COUNT, out, n[axis],
                                               st[axis], n[lo], st[lo], n[hi], st[hi], d[axis]);
    h->launches++;
    return (int)cudaGetLastError();
}

// 1-D density along `axis`.  3-D: a 2-D density first (integrating the cheaper of the other two axes), then a
// second sum; 2-D grids: one sum over the other axis.  scratch: >= the larger 2-D density, DEVICE.
int dbec_launch_density_1d(dbec_handle_s* h, int member, int axis, double* out, double* scratch) {
    const int n[3] = {h->nx, h->ny, h->nz};
    const double d[3] = {h->p.dx, h->p.dy, h->p.dz};
    if (h->p.ndim == 2) {
        const int other = 1 - axis;
        const long long st[2] = {1, h->nx};
        int nblk = (n[axis] + 255) / 256;
        k_density_sum<<<nblk, 256, 0, h->stream>>>(h->psi + (size_t)member * h->P, h->scal + (size_t)member * SC_COUNT, out,
                                                   n[other], st[other], n[axis], st[axis], 1, 0, d[other]);
        h->launches++;
        return (int)cudaGetLastError();
    }
    // integrate first over an axis that is not x unless x is the target's only companion (keeps loads coalesced)
    const int first = axis == 2 ? 1 : 2;                 // x: z then y; y: z then x; z: y then x
    int rc = dbec_launch_density_2d(h, member, first, scratch);
    if (rc) return rc;
    const int lo = first == 0 ? 1 : 0, hi = first == 2 ? 1 : 2;     // scratch is [hi][lo]
    const int second = 3 - axis - first;
    // sum scratch over `second`, keep `axis`
    const long long s_lo = 1, s_hi = n[lo];
    const long long st_axis = axis == lo ? s_lo : s_hi, st_second = second == lo ? s_lo : s_hi;
    int nblk = (n[axis] + 255) / 256;
    k_reduce_rows<<<nblk, 256, 0, h->stream>>>(scratch, out, n[second], st_second, n[axis], st_axis, d[second]);
    h->launches++;
    return (int)cudaGetLastError();
}
