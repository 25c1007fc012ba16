// kernels_small.cu — the WHOLE SSCN step of a small grid in ONE launch, run by ONE thread-block cluster
// ("launching of all required kernels would create a sizeable overhead").
//
// A grid of up to 64 Ki points (BASELINE.json's 32^3 config: psi is 512 KiB) cannot feed 148 SMs, and seven launches
// per step cost more than their work.  Here a cluster of CS CTAs (16 or 8, one per SM) owns a simulation for as many steps
// as dbec_step asks: the data stays in L2, the kernel boundaries of the step become hardware cluster barriers
// (barrier.cluster, release/acquire), and the passes that share an xy plane run back to back in shared memory:
//   A  per plane:   n = |s psi|^2 -> FFT-x (two real lines per transform) -> FFT-y -> spectrum
//   B  per column:  FFT-z, x V_dd(k)/P, inverse FFT-z                                  (calcpsidd2)
//   C  per plane:   inverse FFT-y -> inverse FFT-x -> calcnu -> calclux -> calcluy
//   D  per column:  calcluz, partial sums of calcnorm; the norm factor by a fixed-order sum over the CTAs' partials
//                   read through distributed shared memory
// (2-D grids: a "plane" is one pair of x lines, B and D run along y.)  Four cluster barriers per step, no launch,
// no HBM traffic.  A batch (dbec_create_batch) gives every member its own cluster.  Line lengths are run-time
// numbers (fft_gen.cuh, chunked Thomas with a padded last chunk as in kernels_gen.cu), so every small grid the
// library accepts runs here.  Same arithmetic as the multi-launch path; results agree with it to round-off.
#include <cooperative_groups.h>
#include <algorithm>
#include "dbec_internal.hpp"
#include "fft_gen.cuh"
#include "cn_chunk.cuh"
#include "cn_line_smem.cuh"
#include "trig.cuh"

namespace cg = cooperative_groups;

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return (int)e_; } while (0)

constexpr int SMT = 512;                       // threads per CTA
constexpr int SM_MAX_POINTS = 65536;           // larger grids are served better by the multi-launch path
constexpr size_t SM_TOTAL_BYTES = 224 * 1024;  // dynamic shared memory of a CTA: planes / tiles, chunk ends, staged tables

struct SmallArgs {
    cd* psi; cd* spec; const double* vdd; double* scal;
    const cd* twx; const cd* twy; const cd* twl;            // exp(-2 pi i j / n) of x, y (3-D) and the last axis
    const double* vx; const double* vy; const double* vz;   // trap potential per axis
    GenPlanP px, py, pl;
    int nx, ny, nz, nxhp, nxh1, ndim, nb, nsteps, imag;
    int nyl;          // rows of one unit of the plane passes: NY (3-D: an xy plane), 2 (2-D: a line pair)
    int nunits;       // units per member: NZ (3-D), NY/2 (2-D)
    int ub;           // units a CTA holds in shared memory at once
    int nl, nchl;     // points / chunks along the last axis (z in 3-D, y in 2-D)
    int nr;           // rows of last-axis columns: NY (3-D), 1 (2-D)
    int wspec, wpsi;  // columns per tile of passes B and D
    int nyf;
    int off_a, off_b, off_e;      // shared memory: FFT buffers A and B, chunk ends (elements; psi planes at 0);
                                  // the twiddle tables of x, y and the last axis follow the chunk ends
    double dt, dV;
    long long P, SP;
};

__device__ __forceinline__ cd ldcg2(const cd* p) { return __ldcg(p); }    // L2 only: other SMs rewrite these lines

// Crank-Nicolson solve (cn_chunk.cuh) of `ncols` lines of n points held in shared memory; column q starts at
// (q / C0) * B1 + (q % C0) * B0, element stride es.  Thread (chunk c, column) with the column index fastest; the
// chunks of a column meet through e0 / e1 (2 * SMT elements).  Returns the thread's sum of |u|^2 (calcnorm).
template <bool RT>
__device__ __forceinline__ double cn_smem(cd* P, int ncols, int n, int nch, int C0, int B0, int B1, int es, const CnTab<RT>& cn,
                                          cd* e0, cd* e1) {
    typedef typename CnCoef<RT>::type CT;
    const int G = SMT / nch;                    // columns per round
    const int colg = threadIdx.x % G, c = threadIdx.x / G, j0 = c * CN_L;
    const FastDiv fC0(C0);
    const cd zero = cmake(0.0, 0.0);
    double acc = 0.0;
    for (int cb = 0; cb < ncols; cb += G) {
        const int q = cb + colg;
        const bool active = c < nch && q < ncols;
        int qq, qr;
        fC0.divmod(active ? q : 0, qq, qr);
        cd* g = P + qq * B1 + qr * B0;
        const int jt = active ? j0 : 0;
        cd u[CN_L];
#pragma unroll
        for (int i = 0; i < CN_L; ++i) u[i] = (active && j0 + i < n) ? g[(j0 + i) * es] : zero;
        const cd lo = (active && j0 > 0) ? g[(j0 - 1) * es] : zero;
        const cd hi = (active && j0 + CN_L < n) ? g[(j0 + CN_L) * es] : zero;
        // (the tables are zero-padded to whole chunks: a padded point has h = 0, solves to 0 and feeds nothing back)
        cn_chunk_forward<CT>(u, lo, hi, cn.kap, cn.h + jt);
        if (c < nch) e0[c * G + colg] = u[CN_L - 1];
        __syncthreads();
        cd din = zero;
        for (int i = 0; i < c && i < nch; ++i) din = cn_fma(cn.pf[i * CN_L + CN_L - 1], din, e0[i * G + colg]);
        cn_chunk_backward<CT>(u, din, cn.h + jt, cn.pf + jt);
        if (c < nch) e1[c * G + colg] = u[0];
        __syncthreads();
        cd uin = zero;
        for (int i = nch - 1; i > c; --i) uin = cn_fma(cn.pb[i * CN_L], uin, e1[i * G + colg]);
        cn_chunk_fix<CT>(u, uin, cn.pb + jt);
        if (active) {
#pragma unroll
            for (int i = 0; i < CN_L; ++i)
                if (j0 + i < n) { g[(j0 + i) * es] = u[i]; acc += cnorm2(u[i]); }
        }
        __syncthreads();
    }
    return acc;
}

// Sum over the block in a fixed order; every thread receives the result.
__device__ __forceinline__ double block_sum_all(double x, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) red[w] = x;
    __syncthreads();
    double t = 0.0;
    for (int i = 0; i < SMT / 32; ++i) t += red[i];
    return t;
}

template <bool RT>
__global__ void __launch_bounds__(SMT, 1)
k_small_step(const __grid_constant__ SmallArgs a, CnTab<RT> cnx_g, CnTab<RT> cny_g, CnTab<RT> cnl_g) {
    extern __shared__ __align__(16) cd ssm[];
    __shared__ double sc[SC_COUNT];             // this member's scalars (dbec_internal.hpp)
    __shared__ double red[SMT / 32];
    __shared__ double cpart;                    // this CTA's part of sum |psi|^2, read by the whole cluster
    cg::cluster_group cluster = cg::this_cluster();
    const int CS = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int cid = (int)(blockIdx.x / CS), ncl = (int)(gridDim.x / CS);
    const int tid = threadIdx.x;
    const int nx = a.nx, ny = a.ny, nxh1 = a.nxh1, nxhp = a.nxhp, nyl = a.nyl, nl = a.nl;
    const int pp = nx + 1;                      // pitch of a psi row in shared memory (odd: conflict-free columns)
    cd* Pb = ssm; cd* A = ssm + a.off_a; cd* B = ssm + a.off_b; cd* e0 = ssm + a.off_e; cd* e1 = e0 + SMT;
    // Everything the passes read at data-dependent or repeated addresses is staged in shared memory once: every
    // cluster barrier is an acquire, which drops the L1 copies of global (and local) data, so a table left in
    // global memory costs an L2 round trip inside each dependent chain of each pass (measured: ~1000 cycles per
    // FFT pass and ~2500 per Crank-Nicolson solve on a 16^3 grid, where the arithmetic is a few hundred).
    typedef typename CnCoef<RT>::type CT;
    const int npx = (nx + CN_L - 1) / CN_L * CN_L, npy = (ny + CN_L - 1) / CN_L * CN_L, npl = (nl + CN_L - 1) / CN_L * CN_L;
    const bool d3 = a.ndim == 3;
    cd* twx = e1 + SMT; cd* twy = twx + nx; cd* twl = twy + (d3 ? ny : 0);
    CT* tcx = (CT*)(twl + nl); CT* tcy = tcx + 3 * npx; CT* tcl = tcy + (d3 ? 3 * npy : 0);
    double* vxs = (double*)(tcl + 3 * npl); double* vys = vxs + nx; double* vzs = vys + ny;
    for (int k = tid; k < nx; k += SMT) { twx[k] = a.twx[k]; vxs[k] = a.vx[k]; }
    for (int k = tid; k < ny; k += SMT) { if (d3) twy[k] = a.twy[k]; vys[k] = a.vy[k]; }
    for (int k = tid; k < a.nz; k += SMT) vzs[k] = a.vz[k];
    for (int k = tid; k < nl; k += SMT) twl[k] = a.twl[k];
    for (int k = tid; k < npx; k += SMT) { tcx[k] = cnx_g.h[k]; tcx[npx + k] = cnx_g.pf[k]; tcx[2 * npx + k] = cnx_g.pb[k]; }
    if (d3) for (int k = tid; k < npy; k += SMT) { tcy[k] = cny_g.h[k]; tcy[npy + k] = cny_g.pf[k]; tcy[2 * npy + k] = cny_g.pb[k]; }
    for (int k = tid; k < npl; k += SMT) { tcl[k] = cnl_g.h[k]; tcl[npl + k] = cnl_g.pf[k]; tcl[2 * npl + k] = cnl_g.pb[k]; }
    CnTab<RT> cnx = cnx_g, cny = cny_g, cnl = cnl_g;
    cnx.h = tcx; cnx.pf = tcx + npx; cnx.pb = tcx + 2 * npx;
    cny.h = tcy; cny.pf = tcy + npy; cny.pb = tcy + 2 * npy;
    cnl.h = tcl; cnl.pf = tcl + npl; cnl.pb = tcl + 2 * npl;
    const FastDiv fnx(nx), fnxh1(nxh1), fny(ny), fone(1);
    const long long ls_spec = a.ndim == 3 ? (long long)ny * nxhp : nxhp;       // last-axis strides
    const long long ls_psi = a.ndim == 3 ? (long long)ny * nx : nx;
    const long long vls = a.ndim == 3 ? (long long)a.nyf * nxhp : nxhp;
    // this CTA's share of the units (planes / line pairs) and of the last-axis columns
    const int upc = (a.nunits + CS - 1) / CS, u_lo = min(a.nunits, rank * upc), u_hi = min(a.nunits, u_lo + upc);
    const int ncs = a.nr * nxh1, qs = (ncs + CS - 1) / CS, qs_lo = min(ncs, rank * qs), qs_hi = min(ncs, qs_lo + qs);
    const int ncp = a.nr * nx, qp = (ncp + CS - 1) / CS, qp_lo = min(ncp, rank * qp), qp_hi = min(ncp, qp_lo + qp);

    for (int mem = cid; mem < a.nb; mem += ncl) {
        cd* psi = a.psi + (size_t)mem * a.P;
        cd* spec = a.spec + (size_t)mem * a.SP;
        double* scal = a.scal + (size_t)mem * SC_COUNT;
        __syncthreads();
        if (tid < SC_COUNT) sc[tid] = scal[tid];
        __syncthreads();
        for (int step = 0; step < a.nsteps; ++step) {
            if (tid == 0) ramp_advance(sc);                                  // reading S26 (G, D are used in pass C)
            // ---------------- A: density -> FFT-x -> (FFT-y) -> spectrum ----------------
            for (int u0 = u_lo; u0 < u_hi; u0 += a.ub) {
                const int nu = min(a.ub, u_hi - u0), nrows = nu * nyl, np = nrows / 2;
                const long long r0 = (long long)u0 * nyl;
                const double s2 = sc[SC_S2];
                const cd* g = psi + r0 * nx;
                for (int idx = tid; idx < np * nx; idx += SMT) {
                    int l, x;
                    fnx.divmod(idx, l, x);
                    const cd p0 = ldcg2(g + (2 * l) * nx + x), p1 = ldcg2(g + (2 * l + 1) * nx + x);
                    A[idx] = cmake(s2 * cnorm2(p0), s2 * cnorm2(p1));
                }
                __syncthreads();
                const cd* z = gen_fft_lines2<-1, false>(A, B, np, fone, FastDiv(np), nx, 0, 1, a.px, twx);
                cd* o = (z == A) ? B : A;
                for (int idx = tid; idx < np * nxh1; idx += SMT) {
                    int l, k;
                    fnxh1.divmod(idx, l, k);
                    const cd zk = z[l * nx + k], zp = z[l * nx + (k ? nx - k : 0)];
                    // X_a = (Z[k] + conj Z[N-k])/2,  X_b = (Z[k] - conj Z[N-k])/(2i)
                    o[(2 * l) * nxh1 + k] = cmake(0.5 * (zk.x + zp.x), 0.5 * (zk.y - zp.y));
                    o[(2 * l + 1) * nxh1 + k] = cmake(0.5 * (zk.y + zp.y), -0.5 * (zk.x - zp.x));
                }
                __syncthreads();
                const cd* r = o;
                if (a.ndim == 3) r = gen_fft_lines2<-1, true>(o, (cd*)z, nu * nxh1, FastDiv(nu * nxh1), fnxh1, 1, ny * nxh1, nxh1, a.py, twy);
                cd* gs = spec + r0 * nxhp;
                for (int idx = tid; idx < nrows * nxh1; idx += SMT) {
                    int row, k;
                    fnxh1.divmod(idx, row, k);
                    gs[row * nxhp + k] = r[idx];
                }
                __syncthreads();
            }
            cluster.sync();
            // ---------------- B: last axis forward, x V_dd(k)/P, inverse ----------------
            for (int t0 = qs_lo; t0 < qs_hi; t0 += a.wspec) {
                const int w = min(a.wspec, qs_hi - t0);
                const FastDiv fw(w);
                for (int idx = tid; idx < nl * w; idx += SMT) {
                    int j, c, y, k;
                    fw.divmod(idx, j, c);
                    fnxh1.divmod(t0 + c, y, k);
                    A[idx] = ldcg2(spec + (long long)j * ls_spec + y * nxhp + k);
                }
                __syncthreads();
                cd* r = gen_fft_lines2<-1, true>(A, B, w, fw, fw, 1, 0, w, a.pl, twl);
                cd* o = (r == A) ? B : A;
                for (int idx = tid; idx < nl * w; idx += SMT) {
                    int j, c, y, k;
                    fw.divmod(idx, j, c);
                    fnxh1.divmod(t0 + c, y, k);
                    // folded table (dbec_internal.hpp): index m and N - m share an entry
                    const long long base = a.ndim == 3 ? (long long)(y < ny - y ? y : ny - y) * nxhp + k : k;
                    r[idx] = cmul(a.vdd[base + (long long)(j < nl - j ? j : nl - j) * vls], r[idx]);
                }
                __syncthreads();
                r = gen_fft_lines2<+1, true>(r, o, w, fw, fw, 1, 0, w, a.pl, twl);
                for (int idx = tid; idx < nl * w; idx += SMT) {
                    int j, c, y, k;
                    fw.divmod(idx, j, c);
                    fnxh1.divmod(t0 + c, y, k);
                    spec[(long long)j * ls_spec + y * nxhp + k] = r[idx];
                }
                __syncthreads();
            }
            cluster.sync();
            // ---------------- C: (inverse FFT-y) -> inverse FFT-x -> calcnu -> calclux -> (calcluy) ----------------
            for (int u0 = u_lo; u0 < u_hi; u0 += a.ub) {
                const int nu = min(a.ub, u_hi - u0), nrows = nu * nyl, np = nrows / 2;
                const long long r0 = (long long)u0 * nyl;
                const cd* gs = spec + r0 * nxhp;
                cd* gp = psi + r0 * nx;
                for (int idx = tid; idx < nrows * nxh1; idx += SMT) {
                    int row, k;
                    fnxh1.divmod(idx, row, k);
                    A[idx] = ldcg2(gs + row * nxhp + k);
                }
                for (int idx = tid; idx < nrows * nx; idx += SMT) {
                    int row, x;
                    fnx.divmod(idx, row, x);
                    Pb[row * pp + x] = ldcg2(gp + idx);
                }
                __syncthreads();
                cd* r = A;
                if (a.ndim == 3) r = gen_fft_lines2<+1, true>(A, B, nu * nxh1, FastDiv(nu * nxh1), fnxh1, 1, ny * nxh1, nxh1, a.py, twy);
                cd* o = (r == A) ? B : A;
                for (int idx = tid; idx < np * nx; idx += SMT) {
                    int l, k;
                    fnx.divmod(idx, l, k);
                    const cd* ra = r + (2 * l) * nxh1;
                    const cd* rb = ra + nxh1;
                    cd v;
                    if (k <= nx / 2) { const cd p = ra[k], q = rb[k]; v = cmake(p.x - q.y, p.y + q.x); }         // X_a + i X_b
                    else { const cd p = ra[nx - k], q = rb[nx - k]; v = cmake(p.x + q.y, q.x - p.y); }           // conjugates
                    o[idx] = v;
                }
                __syncthreads();
                const cd* f = gen_fft_lines2<+1, false>(o, r, np, fone, FastDiv(np), nx, 0, 1, a.px, twx);   // (Phi line 2l, Phi line 2l+1)
                {
                    const double s = sc[SC_S], s2 = sc[SC_S2], G = sc[SC_G], D = sc[SC_D], dt = a.dt;
                    for (int idx = tid; idx < nrows * nx; idx += SMT) {
                        int row, x, y, zz;
                        fnx.divmod(idx, row, x);
                        fny.divmod((int)r0 + row, zz, y);
                        const cd ph = f[(row >> 1) * nx + x];
                        const cd q = Pb[row * pp + x];
                        const double u = dt * (vxs[x] + vys[y] + vzs[zz] + G * (s2 * cnorm2(q)) + D * ((row & 1) ? ph.y : ph.x));
                        cd w;
                        if (RT) { double sn, cs; sincos_cw(u, &sn, &cs); w = cmul(s, cmul(q, cmake(cs, -sn))); }
                        else w = cmul(s * exp_cw(-u), q);
                        Pb[row * pp + x] = w;
                    }
                }
                __syncthreads();
                cn_smem<RT>(Pb, nrows, nx, (nx + CN_L - 1) / CN_L, nrows, pp, 0, 1, cnx, e0, e1);
                if (a.ndim == 3) cn_smem<RT>(Pb, nu * nx, ny, (ny + CN_L - 1) / CN_L, nx, 1, ny * pp, pp, cny, e0, e1);
                for (int idx = tid; idx < nrows * nx; idx += SMT) {
                    int row, x;
                    fnx.divmod(idx, row, x);
                    gp[idx] = Pb[row * pp + x];
                }
                __syncthreads();
            }
            cluster.sync();
            // ---------------- D: last-axis sweep (+ calcnorm) ----------------
            double acc = 0.0;
            for (int t0 = qp_lo; t0 < qp_hi; t0 += a.wpsi) {
                const int w = min(a.wpsi, qp_hi - t0);
                const FastDiv fw(w);
                for (int idx = tid; idx < nl * w; idx += SMT) {
                    int j, c;
                    fw.divmod(idx, j, c);
                    Pb[idx] = ldcg2(psi + (long long)j * ls_psi + t0 + c);
                }
                __syncthreads();
                acc += cn_smem<RT>(Pb, w, nl, a.nchl, w, 1, 0, w, cnl, e0, e1);
                for (int idx = tid; idx < nl * w; idx += SMT) {
                    int j, c;
                    fw.divmod(idx, j, c);
                    psi[(long long)j * ls_psi + t0 + c] = Pb[idx];
                }
                __syncthreads();
            }
            if (a.imag) {
                const double part = block_sum_all(acc, red);
                if (tid == 0) cpart = part;
            }
            cluster.sync();
            if (a.imag) {
                // calcnorm (reading S13): the CTAs' partial sums in rank order, the same in every CTA
                if (tid == 0) {
                    double tot = 0.0;
                    for (int r = 0; r < CS; ++r) tot += *cluster.map_shared_rank(&cpart, r);
                    const double sf = 1.0 / sqrt(tot * a.dV);
                    sc[SC_S] = sf; sc[SC_S2] = sf * sf;
                }
                __syncthreads();
            }
        }
        // the member's scalars back to global memory (norm factor, ramp state)
        __syncthreads();
        if (rank == 0 && tid < SC_COUNT) scal[tid] = sc[tid];
        cluster.sync();         // nobody leaves (or overwrites cpart) while a neighbour may still read it
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
static GenPlanP plan_for(int n) {
    GenPlan pl;
    pl.n = n;
    for (int i = 0; i < 12; ++i) pl.fac[i] = 0;
    pl.nfac = n > 1 ? dbec_gen_factor(n, pl.fac) : 0;
    GenPlanP pp;
    make_plan_p(pl, &pp);
    return pp;
}

struct SmallShape { int nyl, nunits, ub, nl, nr, wspec, wpsi, off_a, off_b, off_e; size_t smem; };

// Split n items into equal rounds of at most `most` items: the round size.
static int even_rounds(int n, size_t most) {
    if (most < 1) return 0;
    const int rounds = (int)((n + most - 1) / most);
    return rounds < 1 ? 1 : (n + rounds - 1) / rounds;
}

// Shared-memory plan for `cs` CTAs per cluster; returns false when a single unit does not fit.
// Layout (elements): psi planes or a pass-D tile | FFT buffer A | FFT buffer B | chunk ends (2 * SMT) | constants
// (twiddles, Crank-Nicolson tables — counted as complex in either time mode — trap tables, the three FFT plans).
static bool small_shape(const dbec_handle_s* h, int cs, SmallShape* s) {
    const int nx = h->nx, ny = h->ny, nxh1 = nx / 2 + 1;
    const bool d3 = h->p.ndim == 3;
    s->nyl = d3 ? ny : 2;
    s->nunits = d3 ? h->nz : ny / 2;
    s->nl = d3 ? h->nz : ny;
    s->nr = d3 ? ny : 1;
    const size_t pad16 = CN_L - 1;
    const size_t consts = (size_t)nx + (d3 ? ny : 0) + s->nl + 3 * ((nx + pad16) + (d3 ? ny + pad16 : 0) + (s->nl + pad16)) +
                          (nx + ny + h->nz + 4) / 2 + 3 * (sizeof(GenPlanP) + 15) / 16 + 4;
    const size_t total = SM_TOTAL_BYTES / sizeof(cd);
    if (consts + 2 * SMT >= total) return false;
    const size_t cap = total - consts - 2 * SMT;                         // elements for planes / tiles
    const size_t unit = (size_t)s->nyl * (nx + 1 + 2 * nxh1);
    if (unit > cap || (size_t)3 * s->nl > cap) return false;
    s->ub = even_rounds((s->nunits + cs - 1) / cs, cap / unit);
    size_t pbs = (size_t)s->ub * s->nyl * (nx + 1), ab = (size_t)s->ub * s->nyl * nxh1;
    const int qs = (s->nr * nxh1 + cs - 1) / cs, qp = (s->nr * nx + cs - 1) / cs;
    // passes B and D live in the same buffers: tiles as wide as those allow, at least one column
    s->wspec = even_rounds(qs, std::max<size_t>(1, ab / s->nl));
    s->wpsi = even_rounds(qp, std::max<size_t>(1, pbs / s->nl));
    ab = std::max(ab, (size_t)s->wspec * s->nl);
    pbs = std::max(pbs, (size_t)s->wpsi * s->nl);
    s->off_a = (int)pbs; s->off_b = (int)(pbs + ab); s->off_e = (int)(pbs + 2 * ab);
    s->smem = (pbs + 2 * ab + 2 * SMT + consts) * sizeof(cd);
    return s->smem <= SM_TOTAL_BYTES;
}

static int shape_ok(const dbec_handle_s* h, int cs, SmallShape* s) {
    if (h->P > SM_MAX_POINTS) return 0;
    if (h->p.ndim == 3 && (h->ny % 2)) return 0;             // the line pairs of pass A must not straddle planes
    if (h->nx > DBEC_MAX_N || h->ny > DBEC_MAX_N || h->nz > DBEC_MAX_N) return 0;
    return small_shape(h, cs, s) ? 1 : 0;
}

template <bool RT> static int max_clusters(int cs, size_t smem) {
    auto k = k_small_step<RT>;
    if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    if (cs > 8 && cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) { cudaGetLastError(); return 0; }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cs); cfg.blockDim = dim3(SMT); cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, k, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
    return n;
}

// CTAs per cluster of the one-launch step on this handle, 0 = use the multi-launch path.  request < 0: decide
// here — 3-D grids of up to 64 Ki points whose members all get a resident cluster of their own, 16 CTAs each if
// that many clusters fit, else 8 (measured on B200: 32^3 takes 30 us per step with 16 CTAs, 40 with 8, 49 through
// the seven launches; 2-D grids have four launches per step and stay faster there).  request > 0: that cluster
// size whenever the grid fits (tests).
int dbec_small_choose(dbec_handle_s* h, int request) {
    h->small_max_clusters = 0;
    if (request == 0) return 0;
    const bool rt = h->p.time_mode == 1;
    SmallShape s;
    if (request > 0) {
        if (!shape_ok(h, request, &s)) return 0;
        const int n = rt ? max_clusters<true>(request, s.smem) : max_clusters<false>(request, s.smem);
        if (n < 1) return 0;
        h->small_max_clusters = n;
        return request;
    }
    if (h->p.ndim != 3) return 0;
    for (int cs = 16; cs >= 8; cs >>= 1) {
        if (!shape_ok(h, cs, &s)) continue;
        const int n = rt ? max_clusters<true>(cs, s.smem) : max_clusters<false>(cs, s.smem);
        if (n >= h->nb) { h->small_max_clusters = n; return cs; }
    }
    return 0;
}

template <bool RT> static int launch_small(dbec_handle_s* h, int nsteps) {
    const int cs = h->use_cluster;
    SmallShape s;
    if (!small_shape(h, cs, &s)) return (int)cudaErrorInvalidValue;
    const bool d3 = h->p.ndim == 3;
    SmallArgs a;
    a.psi = h->psi; a.spec = h->spec; a.vdd = h->vdd; a.scal = h->scal;
    a.twx = h->ax[0].twN; a.twy = h->ax[1].twN; a.twl = d3 ? h->ax[2].twN : h->ax[1].twN;
    a.vx = h->ax[0].vtrap; a.vy = h->ax[1].vtrap; a.vz = h->ax[2].vtrap;
    a.px = plan_for(h->nx); a.py = plan_for(h->ny); a.pl = plan_for(s.nl);
    a.nx = h->nx; a.ny = h->ny; a.nz = h->nz; a.nxhp = h->nxhp; a.nxh1 = h->nx / 2 + 1; a.ndim = h->p.ndim; a.nb = h->nb;
    a.nsteps = nsteps; a.imag = h->p.time_mode == 0;
    a.nyl = s.nyl; a.nunits = s.nunits; a.ub = s.ub; a.nl = s.nl; a.nchl = (s.nl + CN_L - 1) / CN_L; a.nr = s.nr;
    a.wspec = s.wspec; a.wpsi = s.wpsi; a.nyf = h->nyf;
    a.off_a = s.off_a; a.off_b = s.off_b; a.off_e = s.off_e;
    a.dt = h->p.dt; a.dV = h->dV; a.P = h->P; a.SP = h->SP;
    auto k = k_small_step<RT>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s.smem));
    if (cs > 8) CK(cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(SMT);
    cfg.dynamicSmemBytes = s.smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    // (clusters that can be resident at once, from dbec_small_choose: more would only queue up behind them)
    const int ncl = h->nb < h->small_max_clusters ? h->nb : h->small_max_clusters;
    cfg.gridDim = dim3(cs * ncl);
    const CnTab<RT> cx = make_cntab<RT>(h->ax[0]), cy = make_cntab<RT>(h->ax[1]), cl = make_cntab<RT>(h->ax[d3 ? 2 : 1]);
    CK(cudaLaunchKernelEx(&cfg, k, a, cx, cy, cl));
    h->launches++;
    return (int)cudaGetLastError();
}

int dbec_launch_small_step(dbec_handle_s* h, int nsteps) {
    if (h->use_small_p2) return dbec_launch_small_p2(h, nsteps);
    return h->p.time_mode == 1 ? launch_small<true>(h, nsteps) : launch_small<false>(h, nsteps);
}
