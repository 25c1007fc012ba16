// kernels_xline.cu — the passes along x (contiguous grid lines) as persistent, warp-specialised
// sm_100a kernels fed by bulk asynchronous copies (cp.async.bulk + mbarrier, tma_pipe.cuh):
//
//   k_xline_nonlin   a3 along x (complex-to-real inverse FFT, two real lines per complex transform,
//                    PAPER.md:71) + a4 psi <- s psi exp(-c dt (V + G n + D Phi)) (calcnu)
//                    + a5 the Crank-Nicolson sweep along x (calclux), one tile of
//                    8 grid lines at a time, all in shared memory.
//   k_xline_density  a1 along x: n = |s psi|^2 fused into the forward real-to-complex transform.
//
// Same arithmetic as k_ifftx_nonlin / k_density_fftx (kernels_fft.cu); what changes is that the next
// tiles' loads and the previous tiles' stores are in flight while a tile is being worked on.
#include "dbec_internal.hpp"
#include "fft_line.cuh"
#include "cn_chunk.cuh"
#include "cn_line_smem.cuh"
#include "tma_pipe.cuh"
#include "trig.cuh"

// calcnu: points evaluated side by side (8 measures slower than 4)
constexpr int NLU_C = 4;
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return (int)e_; } while (0)

// XP line pairs (XR = 2 XP grid lines) per tile: 4 pairs up to 256 points, 2 pairs of 512 points
template <int N> struct XPlan;
template <> struct XPlan<128> { typedef FftPlan<8, 1, true> P;  static constexpr int XP = 4; };
template <> struct XPlan<256> { typedef FftPlan<16, 1, true> P; static constexpr int XP = 4; };
template <> struct XPlan<512> { typedef FftPlan<16, 2, true> P; static constexpr int XP = 2; };

__host__ __device__ constexpr int nxhp_of(int n) { return ((n / 2 + 1) + DBEC_SPEC_COLS - 1) / DBEC_SPEC_COLS * DBEC_SPEC_COLS; }

// ------------------------------------------------------------------------------------------------
// a3 (x) + a4 + a5
// ------------------------------------------------------------------------------------------------
// Stage layout: 8 psi lines with a pitch of N+1 elements (so that the 8 lines of a tile sit in 8
// different 16-byte bank groups and the chunked Thomas pass reads them without conflicts), then the
// 8 half-spectrum rows.  A pair's two spectrum rows (2*NXHP elements) double as its FFT exchange
// buffer once they are in registers; after the transform the spectrum area holds the chunk ends of
// the Thomas carries.
template <class P, int XP, bool RT, int NG, int NST>
__global__ void __launch_bounds__(NG * 2 * XP * P::T + 96, 1)
k_xline_nonlin(const cd* __restrict__ spec, cd* __restrict__ psi, const cd* __restrict__ twA_g,
               const cd* __restrict__ twN_g, const double* __restrict__ scal, const double* __restrict__ vx_g,
               const double* __restrict__ vy, const double* __restrict__ vz, double dt, int ntiles, int ny, int nz,
               int nb, long long row0, CnTab<RT> cn, int rev, float pol_ld, float pol_st, float pol_spec) {
    typedef typename CnCoef<RT>::type CT;
    // A group of GT = 8*T threads owns one tile: its first half runs the four pair transforms (T threads
    // per pair), then all of it runs calcnu (T threads per line) and calclux (one 16-point chunk each).
    constexpr int XR = 2 * XP;
    constexpr int T = P::T, N = P::N, NCH = N / CN_L, GT = XR * T, NT = NG * GT + 96;
    constexpr int NXHP = nxhp_of(N), PITCH = N + 1;
    // a pair's area: its two spectrum rows, later its FFT exchange, later Phi as two real lines
    constexpr int SPP = (P::SMEM > 2 * NXHP) ? P::SMEM : 2 * NXHP;
    constexpr int PSI_BYTES = XR * PITCH * (int)sizeof(cd), SPEC_BYTES = XP * SPP * (int)sizeof(cd);
    constexpr int STAGE_BYTES = PSI_BYTES + SPEC_BYTES;
    constexpr int E = cn_tab_elems(N);
    static_assert(NCH == T, "one chunk per thread of a line");
    static_assert(2 * NCH * XR <= XP * SPP, "chunk ends must fit the spectrum area");
    extern __shared__ __align__(1024) unsigned char smraw[];
    unsigned char* base = smraw;     // (no integer round trip: the compiler must see shared-memory pointers)
    cd* tw = (cd*)(base + (size_t)NST * STAGE_BYTES);            // twA [N], twN [N]
    CT* tab = (CT*)(tw + 2 * N);                                 // h, PF, PB (padded), PFE, PBS
    double* vxs = (double*)(tab + 3 * E + 2 * NCH);              // trap table along x
    uint64_t* bars = (uint64_t*)(vxs + N);
    uint64_t* full = bars; uint64_t* empty = bars + NST; uint64_t* done = bars + 2 * NST;
    int* issued = (int*)(bars + 3 * NST);
    const int tid = threadIdx.x;
    for (int k = tid; k < N; k += NT) { tw[k] = twA_g[k]; tw[N + k] = twN_g[k]; vxs[k] = dt * vx_g[k]; }
    CnTab<RT> cs = cn_stage_tables<RT, N>(cn, tab);
    for (int k = tid; k < NCH; k += NT) { tab[3 * E + k] = cn.pfe[k]; tab[3 * E + NCH + k] = cn.pbs[k]; }
    cs.pfe = tab + 3 * E; cs.pbs = tab + 3 * E + NCH;
    if (tid == 0) {
        *issued = 0;
        for (int s = 0; s < NST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); mbar_init(done + s, GT / 32); }
        fence_mbar_init();
    }
    __syncthreads();
    pdl_launch_dependents();        // the next kernel of the stream may start its own prologue
    pdl_wait();                     // tables are staged, barriers set up: now wait for the previous kernel's data
    const int nmine = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    if (tid < NG * GT) {
        const int g = tid / GT, t = tid % GT;
        const int lp = t / T, m = t % T;                 // transform: pair lp (t < GT/2); calcnu: line lp, x = j*T + m
        const int r = t % XR, c = t / XR;                // calclux: line r, chunk c
        const cd* twA = tw; const cd* twN = tw + N;
        // u = dt V + dtG |q|^2 + dtD Phi; the scalars belong to the tile's batch member (one member: loaded once)
        double s = scal[SC_S];
        double dtG = dt * (scal[SC_G] * scal[SC_S2]), dtD = dt * scal[SC_D];
        // trap potential of this thread's line, V_y + V_z, fetched one tile ahead (global tables)
        auto row_of = [&](int i) {
            long long tile = (long long)blockIdx.x + (long long)i * gridDim.x;
            if (rev) tile = ntiles - 1 - tile;
            return (int)(row0 + tile * XR) + lp;
        };
        auto vrow_of = [&](int i) {
            const int row = row_of(i);
            return dt * (vy[row % ny] + vz[(row / ny) % nz]);
        };
        double vrow = (g < nmine) ? vrow_of(g) : 0.0;
        for (int i = g; i < nmine; i += NG) {
            const int st = i % NST;
            const double vrow_next = (i + NG < nmine) ? vrow_of(i + NG) : 0.0;
            if (nb > 1) {
                const double* sc = scal + (size_t)(row_of(i) / (ny * nz)) * SC_COUNT;
                s = sc[SC_S]; dtG = dt * (sc[SC_G] * sc[SC_S2]); dtD = dt * sc[SC_D];
            }
            wait_issued(issued, i);
            mbar_wait(full + st, (i / NST) & 1);
            cd* ps = (cd*)(base + (size_t)st * STAGE_BYTES);
            cd* ss = (cd*)(base + (size_t)st * STAGE_BYTES + PSI_BYTES);
            // ---- inverse transform of a pair's spectrum: v[j] = (Phi on line a, Phi on line b) at x = j*T + m;
            //      Phi goes back to the pair's spectrum rows as two real lines [2][N]
            if (t < GT / 2) {
                cd* sa = ss + lp * SPP;
                const cd* sb = sa + NXHP;
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
                __syncwarp();                                        // the pair's rows are in registers: reuse them
                fft_line<P, +1, 0>(v, m, sa, 1, twA, twN);
                __syncwarp();
                double* ph = (double*)sa;
#pragma unroll
                for (int j = 0; j < 16; ++j) { ph[j * T + m] = v[j].x; ph[N + j * T + m] = v[j].y; }
            }
            named_bar_sync(1 + g, GT);
            // ---- calcnu on line lp
            {
                cd* p = ps + lp * PITCH;
                const double* ph = (const double*)(ss + (lp >> 1) * SPP) + (lp & 1) * N;
                // NLU_C points at a time, all their loads first and all their stores last: p, ph and vxs point
                // into the same shared array, so a store in between would pin every later load behind it and
                // the evaluations would run one after the other (8-cycle fp64 latency, ~30 dependent steps each)
#pragma unroll 1
                for (int j0 = 0; j0 < 16; j0 += NLU_C) {
                    cd q[NLU_C];
                    double u[NLU_C];
#pragma unroll
                    for (int jj = 0; jj < NLU_C; ++jj) {
                        const int x = (j0 + jj) * T + m;
                        q[jj] = p[x];
                        u[jj] = fma(dtD, ph[x], vxs[x] + vrow);
                    }
#pragma unroll
                    for (int jj = 0; jj < NLU_C; ++jj) {
                        u[jj] = fma(dtG, cnorm2(q[jj]), u[jj]);
                        if (RT) {
                            double sn, cs_;
                            sincos_cw(u[jj], &sn, &cs_);          // branch-free: the evaluations interleave
                            q[jj] = cmul(s, cmul(q[jj], cmake(cs_, -sn)));
                        } else {
                            q[jj] = cmul(s * exp_cw(-u[jj]), q[jj]);
                        }
                    }
#pragma unroll
                    for (int jj = 0; jj < NLU_C; ++jj) p[(j0 + jj) * T + m] = q[jj];
                }
            }
            named_bar_sync(1 + g, GT);
            // ---- calclux: line r, chunk c
            cd* line = ps + r * PITCH + c * CN_L;
            cd* e0 = ss;                    // [NCH][XR] forward chunk ends
            cd* e1 = ss + NCH * XR;         // [NCH][XR] backward chunk starts
            cd u[CN_L];
#pragma unroll
            for (int k = 0; k < CN_L; ++k) u[k] = line[k];
            const cd lo = (c > 0) ? line[-1] : cmake(0.0, 0.0);
            const cd hi = (c < NCH - 1) ? line[CN_L] : cmake(0.0, 0.0);
            cn_chunk_forward<CT>(u, lo, hi, cs.kap, cs.h + 17 * c);
            e0[c * XR + r] = u[CN_L - 1];
            named_bar_sync(1 + g, GT);
            const cd din = cn_carry_forward<CT>(c, e0 + r, XR, cs.pfe, cs.K);
            cn_chunk_backward<CT>(u, din, cs.h + 17 * c, cs.pf + 17 * c);
            e1[c * XR + r] = u[0];
            named_bar_sync(1 + g, GT);
            const cd uin = cn_carry_backward<CT>(c, NCH, e1 + r, XR, cs.pbs, cs.K);
            cn_chunk_fix<CT>(u, uin, cs.pb + 17 * c);
#pragma unroll
            for (int k = 0; k < CN_L; ++k) line[k] = u[k];
            fence_proxy_async();
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(done + st);
            vrow = vrow_next;
        }
    } else if (tid == NG * GT) {
        const uint64_t pol = l2_policy_code(pol_spec), polp = l2_policy_code(pol_ld);
        for (int i = 0; i < nmine; ++i) {
            const int st = i % NST;
            if (i >= NST) mbar_wait(empty + st, ((i / NST) - 1) & 1);
            st_release_shared(issued, i + 1);
            mbar_expect_tx(full + st, XR * N * (int)sizeof(cd) + XR * NXHP * (int)sizeof(cd));
            long long tile = (long long)blockIdx.x + (long long)i * gridDim.x;
            if (rev) tile = ntiles - 1 - tile;
            unsigned char* dst = base + (size_t)st * STAGE_BYTES;
            const cd* src = psi + tile * XR * N;
#pragma unroll 1
            for (int rr = 0; rr < XR; ++rr)
                bulk_load_hint(dst + (size_t)rr * PITCH * sizeof(cd), src + (size_t)rr * N, N * (int)sizeof(cd), full + st, polp);
#pragma unroll 1
            for (int pp = 0; pp < XP; ++pp)
                bulk_load_hint(dst + PSI_BYTES + (size_t)pp * SPP * sizeof(cd), spec + (tile * XP + pp) * 2 * NXHP,
                               2 * NXHP * (int)sizeof(cd), full + st, pol);
        }
    } else if (tid == NG * GT + 32 || tid == NG * GT + 64) {
        // two storers (even / odd stages): while one sits in wait_group.read (which lasts about as long
        // as the global write), the other already drains the next finished stage
        const int which = (tid - NG * GT) / 32 - 1;      // storer 0: even stages, storer 1: odd stages
        const uint64_t polp = l2_policy_code(pol_st);
        for (int i = 0; i < nmine; ++i) {
            const int st = i % NST;
            if ((st & 1) != which) continue;
            mbar_wait(done + st, (i / NST) & 1);
            long long tile = (long long)blockIdx.x + (long long)i * gridDim.x;
            if (rev) tile = ntiles - 1 - tile;
            const unsigned char* src = base + (size_t)st * STAGE_BYTES;
            cd* dstg = psi + tile * XR * N;
#pragma unroll 1
            for (int rr = 0; rr < XR; ++rr)
                bulk_store_hint(dstg + (size_t)rr * N, src + (size_t)rr * PITCH * sizeof(cd), N * (int)sizeof(cd), polp);
            bulk_commit();
            bulk_wait_read<0>();
            mbar_arrive(empty + st);
        }
        bulk_wait<0>();
    }
}

// ------------------------------------------------------------------------------------------------
// a1 (x): n = |s psi|^2 -> half spectrum along x
// ------------------------------------------------------------------------------------------------
// A stage holds the 8 psi lines of a tile (contiguous, one bulk load).  The T threads of a pair read
// its two lines into registers, then reuse the pair's 2N-element area: [0, 2*NXHP) FFT exchange, later
// the pair's two output rows; [N, 2N) the transform Z, of which other threads read only the upper half
// (the mirror Z[N-k], k = 1..N/2).  One bulk store per pair.
template <class P, int XP, int NG, int NST>
__global__ void __launch_bounds__(NG* XP* P::T + 96, 1)
k_xline_density(const cd* __restrict__ psi, cd* __restrict__ spec, const cd* __restrict__ twA_g,
                const cd* __restrict__ twN_g, double* __restrict__ scal, int ntiles, int tiles_per_member, int nb,
                int advance, int rev, float pol_psi, float pol_spec, PaceArgs pace) {
    constexpr int XR = 2 * XP;
    constexpr int T = P::T, N = P::N, GT = XP * T, NT = NG * GT + 96;
    constexpr int NXHP = nxhp_of(N);
    constexpr int STAGE_BYTES = XR * N * (int)sizeof(cd), PAIR_BYTES = 2 * NXHP * (int)sizeof(cd);
    static_assert(P::SMEM <= N + N / 2 && 2 * NXHP <= N + N / 2, "exchange / output rows must stay below Z's upper half");
    extern __shared__ __align__(1024) unsigned char smraw[];
    unsigned char* base = smraw;
    cd* tw = (cd*)(base + (size_t)NST * STAGE_BYTES);
    uint64_t* bars = (uint64_t*)(tw + 2 * N);
    uint64_t* full = bars; uint64_t* empty = bars + NST; uint64_t* done = bars + 2 * NST;
    int* issued = (int*)(bars + 3 * NST);
    const int tid = threadIdx.x;
    for (int k = tid; k < N; k += NT) { tw[k] = twA_g[k]; tw[N + k] = twN_g[k]; }
    if (tid == 0) {
        *issued = 0;
        for (int s = 0; s < NST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); mbar_init(done + s, GT / 32); }
        fence_mbar_init();
    }
    __syncthreads();
    pdl_launch_dependents();        // the next kernel of the stream may start its own prologue
    pdl_wait();                     // tables are staged, barriers set up: now wait for the previous kernel's data
    const int nmine = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    auto tile_of = [&](int i) {
        const long long t = (long long)blockIdx.x + (long long)i * gridDim.x;
        return rev ? (long long)ntiles - 1 - t : t;
    };
    if (tid < NG * GT) {
        const int g = tid / GT, t = tid % GT, lp = t / T, m = t % T;
        const cd* twA = tw; const cd* twN = tw + N;
        double s2 = scal[SC_S2];
        for (int i = g; i < nmine; i += NG) {
            const int st = i % NST;
            if (nb > 1) s2 = scal[(size_t)(tile_of(i) / tiles_per_member) * SC_COUNT + SC_S2];    // the tile's batch member
            wait_issued(issued, i);
            mbar_wait(full + st, (i / NST) & 1);
            cd* pr = (cd*)(base + (size_t)st * STAGE_BYTES) + lp * 2 * N;     // the pair's area
            cd v[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const cd a = pr[j * T + m], b = pr[N + j * T + m];
                v[j] = cmake(s2 * cnorm2(a), s2 * cnorm2(b));
            }
            __syncwarp();
            fft_line<P, -1, 0>(v, m, pr, 1, twA, twN);
            __syncwarp();
#pragma unroll
            for (int j = 8; j < 16; ++j) pr[N + j * T + m] = v[j];            // Z[N/2 .. N-1]
            __syncwarp();
            // mirrors first, stores afterwards (a store in between would pin the later loads behind it)
            cd zm[9];
#pragma unroll
            for (int j = 0; j <= 8; ++j) {
                const int k = j * T + m;
                zm[j] = (k == 0 || k > N / 2) ? v[j] : pr[2 * N - k];         // Z[N-k]
            }
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int k = j * T + m;
                if (k <= N / 2) {
                    const cd z = v[j], zp = zm[j < 9 ? j : 8];
                    // X_a = (Z[k] + conj Z[N-k])/2,  X_b = (Z[k] - conj Z[N-k])/(2i)
                    pr[k] = cmake(0.5 * (z.x + zp.x), 0.5 * (z.y - zp.y));
                    pr[NXHP + k] = cmake(0.5 * (z.y + zp.y), -0.5 * (z.x - zp.x));
                } else if (k < NXHP) {
                    pr[k] = cmake(0.0, 0.0);
                    pr[NXHP + k] = cmake(0.0, 0.0);
                }
            }
            fence_proxy_async();
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(done + st);
        }
    } else if (tid == NG * GT) {
        // first kernel of a step: move the NSTP ramp on (nothing in this kernel reads G or D)
        if (advance && blockIdx.x == 0)
            for (int b = 0; b < nb; ++b) ramp_advance(scal + (size_t)b * SC_COUNT);
        const uint64_t pol = l2_policy_code(pol_psi);
        unsigned long long t0 = 0;
        for (int i = 0; i < nmine; ++i) {
            const int st = i % NST;
            if (i >= NST) mbar_wait(empty + st, ((i / NST) - 1) & 1);
            if (pace.ns) pace_wait(t0, i, pace);
            st_release_shared(issued, i + 1);
            mbar_expect_tx(full + st, STAGE_BYTES);
            bulk_load_hint(base + (size_t)st * STAGE_BYTES, psi + tile_of(i) * XR * N, STAGE_BYTES, full + st, pol);
        }
        if (pace.ns) pace_done(pace.st);
    } else if (tid == NG * GT + 32 || tid == NG * GT + 64) {
        const int which = (tid - NG * GT) / 32 - 1;      // storer 0: even stages, storer 1: odd stages
        for (int i = 0; i < nmine; ++i) {
            const int st = i % NST;
            if ((st & 1) != which) continue;
            mbar_wait(done + st, (i / NST) & 1);
            const unsigned char* src = base + (size_t)st * STAGE_BYTES;
            const uint64_t pols = l2_policy_code(pol_spec);
            cd* dstg = spec + tile_of(i) * XR * NXHP;
#pragma unroll 1
            for (int pp = 0; pp < XP; ++pp)
                bulk_store_hint(dstg + (size_t)pp * 2 * NXHP, src + (size_t)pp * 2 * N * sizeof(cd), PAIR_BYTES, pols);
            bulk_commit();
            bulk_wait_read<0>();
            mbar_arrive(empty + st);
        }
        bulk_wait<0>();
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
int dbec_xline_supported(const dbec_handle_s* h) {
    // (a tile of 8 lines never straddles two batch members: ny * nz is a multiple of 8)
    return h->use_tma && (h->nx == 128 || h->nx == 256 || h->nx == 512) && ((h->ny * h->nz) % 8 == 0);
}

template <int N, bool RT, int NG, int NST, int XP = XPlan<N>::XP> static int launch_xline_nonlin(dbec_handle_s* h, int z0, int nzs) {
    typedef typename XPlan<N>::P P;
    typedef typename CnCoef<RT>::type CT;
    constexpr int XR = 2 * XP;
    constexpr int GT = XR * P::T, NXHP = nxhp_of(N);
    constexpr int SPP = (P::SMEM > 2 * NXHP) ? P::SMEM : 2 * NXHP;
    constexpr int STAGE = XR * (N + 1) * (int)sizeof(cd) + XP * SPP * (int)sizeof(cd);
    if (h->nxhp != NXHP) return (int)cudaErrorInvalidValue;
    const int ntiles = (int)((long long)h->ny * nzs / XR);
    const int grid = ntiles < h->num_sms ? ntiles : h->num_sms;
    const size_t sm = (size_t)NST * STAGE + 2 * N * sizeof(cd) + (3 * cn_tab_elems(N) + 2 * (N / CN_L)) * sizeof(CT) +
                      N * sizeof(double) + (3 * NST + 1) * sizeof(uint64_t);
    auto k = k_xline_nonlin<P, XP, RT, NG, NST>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const long long row0 = (long long)z0 * h->ny;
    CK(launch_pdl(k, dim3(grid), dim3(NG * GT + 96), sm, h->stream, h->use_pdl, h->spec + row0 * NXHP, h->psi + row0 * N, h->ax[0].twA, h->ax[0].twN, h->scal,
                                             h->ax[0].vtrap, h->ax[1].vtrap, h->ax[2].vtrap, h->p.dt, ntiles, h->ny, h->nz, h->nb, row0,
                                             make_cntab<RT>(h->ax[0]), h->rev_next, h->pol[POL_NL_LD], h->pol[POL_NL_ST], h->pol[POL_NL_SPEC]));
    h->launches++;
    return (int)cudaGetLastError();
}

int dbec_launch_xline_nonlin(dbec_handle_s* h, int z0, int nzs) {
    const bool rt = h->p.time_mode == 1;
    switch (h->nx) {
        case 128: return rt ? launch_xline_nonlin<128, true, 4, 8>(h, z0, nzs) : launch_xline_nonlin<128, false, 4, 8>(h, z0, nzs);
        case 256: return rt ? launch_xline_nonlin<256, true, 3, 4>(h, z0, nzs) : launch_xline_nonlin<256, false, 3, 4>(h, z0, nzs);
        case 512: return rt ? launch_xline_nonlin<512, true, 2, 3>(h, z0, nzs) : launch_xline_nonlin<512, false, 2, 3>(h, z0, nzs);
        default: return (int)cudaErrorInvalidValue;
    }
}

template <int N, int NG, int NST> static int launch_xline_density(dbec_handle_s* h, int z0, int nzs, int advance) {
    typedef typename XPlan<N>::P P;
    constexpr int XP = XPlan<N>::XP, XR = 2 * XP;
    constexpr int GT = XP * P::T, NXHP = nxhp_of(N);
    if (h->nxhp != NXHP) return (int)cudaErrorInvalidValue;
    const int ntiles = (int)((long long)h->ny * nzs / XR);
    const int grid = ntiles < h->num_sms ? ntiles : h->num_sms;
    const size_t sm = (size_t)NST * XR * N * sizeof(cd) + 2 * N * sizeof(cd) + (3 * NST + 1) * sizeof(uint64_t);
    auto k = k_xline_density<P, XP, NG, NST>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const long long row0 = (long long)z0 * h->ny;
    CK(launch_pdl(k, dim3(grid), dim3(NG * GT + 96), sm, h->stream, h->use_pdl, h->psi + row0 * N, h->spec + row0 * NXHP, h->ax[0].twA, h->ax[0].twN, h->scal,
                                             ntiles, h->ny * h->nz / XR, h->nb, advance, h->rev_next, h->pol[POL_D_PSI], h->pol[POL_D_SPEC],
                                             dbec_pace_args(h, ntiles, grid, (size_t)XR * (N + NXHP) * sizeof(cd), 16.0 * (double)h->P * h->nb)));
    h->launches++;
    return (int)cudaGetLastError();
}

int dbec_launch_xline_density(dbec_handle_s* h, int z0, int nzs, int advance) {
    switch (h->nx) {
        case 128: return launch_xline_density<128, 4, 12>(h, z0, nzs, advance);
        case 256: return launch_xline_density<256, 4, 6>(h, z0, nzs, advance);
        case 512: return launch_xline_density<512, 4, 6>(h, z0, nzs, advance);
        default: return (int)cudaErrorInvalidValue;
    }
}
