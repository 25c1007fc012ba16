// kernels_xwarp.cu — a3 along x (complex-to-real inverse FFT) + a4 calcnu + a5 calclux
// with ONE WARP PER LINE PAIR: the successor of k_xline_nonlin for lines of 128 and 256 points.
//
// k_xline_nonlin gives a tile of 8 lines to a group of 128 threads and separates its three phases by four
// block-level barriers; ncu (profiles/r2_xline_before.md) puts 23 % of its warp time into those barriers, half of
// the group idles during the pair transforms, and psi crosses shared memory twice.  Here a warp owns its lines
// from the moment they land to the moment they leave:
//   * the pair's spectrum rows -> 8 values per lane -> 256-point inverse FFT inside the warp (fft_linev.cuh:
//     V = 8, T = 32; every exchange is a __syncwarp) -> Phi_dd of both lines, interleaved (a, b), in shared memory;
//   * each lane then takes 8 CONSECUTIVE points of each line: calcnu on them in registers, and the very same
//     registers are one chunk of the Crank-Nicolson solve (cn_chunk.cuh with L = 8).  Neighbour values, the
//     zero-start chunk ends and the carries travel by warp shuffles: no shared-memory round trip, no barrier.
//   * psi lands and leaves through a tensor map with the 128-byte swizzle: a lane's chunk is one 128-byte row,
//     whose 16-byte units the hardware rotates by the row index, so the 32 chunk reads of a warp are
//     conflict-free although they are 128 bytes apart (without the swizzle: 8-way conflicts).
// The carry into a chunk is the Horner sum over ALL earlier chunk ends with the factors pfe (products of L
// consecutive h_j, |h_j| < 1); the host (dbec_api.cu) counts how many terms K are above 2^-73 of the first one
// (3 for BASELINE.json's real-time configs, 2 for the imaginary-time ones) and the kernel sums exactly those:
// the dropped terms are below the last bit of the sum.  Handles whose K exceeds the 31 lanes a shuffle reaches
// stay with k_xline_nonlin.
#include "dbec_internal.hpp"
#include "fft_linev.cuh"
#include "cn_chunk.cuh"
#include "tma_pipe.cuh"
#include "trig.cuh"

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return (int)e_; } while (0)

constexpr int WL = 8;              // Crank-Nicolson chunk: 8 points = one 128-byte row of psi
// calcnu: points evaluated side by side (same reason as NLU_C in kernels_xline.cu); both time modes use the
// branch-free functions of trig.cuh, whose evaluations interleave
template <bool RT> struct NlwBatch { static constexpr int C = 4; };

template <int N> struct WPlan;
template <> struct WPlan<256> { typedef FftPlanV<8, 8, 4> P; };     // one pair per warp (32 lanes)
template <> struct WPlan<128> { typedef FftPlanV<8, 8, 2> P; };     // two pairs per warp (16 lanes each)

__host__ __device__ constexpr int w_nxhp(int n) { return ((n / 2 + 1) + DBEC_SPEC_COLS - 1) / DBEC_SPEC_COLS * DBEC_SPEC_COLS; }
// positions inside the padded rows: a lane's 8 values sit 80 (doubles) / 144 (complex table entries) bytes
// after its neighbour's, so that the 128-bit loads of a quarter warp fall into eight different bank groups
__host__ __device__ constexpr int padd(int k) { return k + 2 * (k >> 3); }          // doubles (Phi, trap)
__host__ __device__ constexpr int padt(int k) { return k + (k >> 3); }              // table entries (h, PF, PB), Phi pairs
// elements of a pair's area: its two spectrum rows, later the FFT exchange, later the padded row of Phi pairs
__host__ __device__ constexpr int w_pair_el(int fft, int nxhp, int ntab) {
    return fft > 2 * nxhp ? (fft > ntab ? fft : ntab) : (2 * nxhp > ntab ? 2 * nxhp : ntab);
}

template <bool RT> struct CnTabW {
    typedef typename CnCoef<RT>::type CT;
    const CT* h; const CT* pf; const CT* pb; const CT* pfe; const CT* pbs;
    CT kap;
    int K;                   // carry terms (see the header)
};

__device__ __forceinline__ cd shfl_up_cd(cd v, int d, int w) {
    return cmake(__shfl_up_sync(0xffffffffu, v.x, d, w), __shfl_up_sync(0xffffffffu, v.y, d, w));
}
__device__ __forceinline__ cd shfl_down_cd(cd v, int d, int w) {
    return cmake(__shfl_down_sync(0xffffffffu, v.x, d, w), __shfl_down_sync(0xffffffffu, v.y, d, w));
}

template <int N, bool RT, int NW, int NST>
__global__ void __launch_bounds__((NW + 3) * 32, 1)
k_xwarp_nonlin(const __grid_constant__ CUtensorMap map_psi, const cd* __restrict__ spec, const cd* __restrict__ twN_g,
               const double* __restrict__ scal, const double* __restrict__ vx_g, const double* __restrict__ vy,
               const double* __restrict__ vz, double dt, int ntiles, int ny, int nz, int nb, CnTabW<RT> cn, int rev,
               float pol_ld, float pol_st, float pol_spec, PaceArgs pace) {
    typedef typename CnCoef<RT>::type CT;
    typedef typename WPlan<N>::P P;
    constexpr int NLW_C = NlwBatch<RT>::C;
    constexpr int T = P::T, PAIRS = 32 / T, LPT = 2 * PAIRS;         // lines per tile (= per warp)
    constexpr int CPL = N / WL;                                      // chunks per line = lanes per line
    constexpr int NXHP = w_nxhp(N);
    constexpr int NTAB = N + N / 8;                                  // padded table / padded Phi row (entries)
    constexpr int PAIR_EL = w_pair_el(P::SMEM, NXHP, NTAB);          // a pair's area: spectrum rows, FFT exchange, Phi
    constexpr int NPD = N + N / 4;                                   // padded real row (doubles)
    constexpr int PSI_BYTES = LPT * N * (int)sizeof(cd), SLOT_BYTES = PAIRS * PAIR_EL * (int)sizeof(cd);
    static_assert(PSI_BYTES % 1024 == 0, "the swizzle pattern needs 1024-byte aligned psi tiles");
    constexpr int NT = (NW + 3) * 32;
    extern __shared__ __align__(1024) unsigned char smraw[];
    unsigned char* base = smraw;     // (no integer round trip: the compiler must see shared-memory pointers)
    unsigned char* slots = base + (size_t)NST * PSI_BYTES;       // psi tiles first (1024-byte aligned), then the pair areas
    cd* tw = (cd*)(slots + (size_t)NST * SLOT_BYTES);            // twA [N] (stage-1 twiddles), tw2 [R3*R2] (stage 2)
    CT* tab = (CT*)(tw + N + P::T);                              // h, PF, PB (padded), PFE, PBS
    double* vxs = (double*)(tab + 3 * NTAB + 2 * CPL);           // dt * trap along x (padded)
    uint64_t* bars = (uint64_t*)(vxs + NPD);
    uint64_t* full = bars; uint64_t* empty = bars + NST; uint64_t* done = bars + 2 * NST;
    int* issued = (int*)(bars + 3 * NST);
    const int tid = threadIdx.x;
    for (int k = tid; k < N; k += NT) {
        tw[k] = twN_g[((k % T) * (k / T)) % N];                  // twA[k1*T + m] = W_N^{m k1}
        if (k < T) tw[N + k] = twN_g[(P::V * (k % P::R3) * (k / P::R3)) % N];   // tw2[k2*R3 + n3] = W_N^{V n3 k2}
        vxs[padd(k)] = dt * vx_g[k];
        tab[padt(k)] = cn.h[k]; tab[NTAB + padt(k)] = cn.pf[k]; tab[2 * NTAB + padt(k)] = cn.pb[k];
    }
    for (int k = tid; k < CPL; k += NT) { tab[3 * NTAB + k] = cn.pfe[k]; tab[3 * NTAB + CPL + k] = cn.pbs[k]; }
    if (tid == 0) {
        *issued = 0;
        for (int s = 0; s < NST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); mbar_init(done + s, 1); }
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
    const int warp = tid >> 5, lane = tid & 31;
    if (warp < NW) {
        const cd* twA = tw; const cd* tw2 = tw + N;
        const CT* th = tab; const CT* tpf = tab + NTAB; const CT* tpb = tab + 2 * NTAB;
        const CT* pfe = tab + 3 * NTAB; const CT* pbs = pfe + CPL;
        const CT kap = cn.kap;
        const int K = cn.K;
        const int m = lane % T, pr = lane / T;                   // FFT: lane m of pair pr
        const int c = lane % CPL, sub = lane / CPL;              // calcnu + calclux: chunk c of line 2*slot*?+sub (below)
        // slot s of this lane: line ls[s] of the tile.  N = 256: the two lines of the pair (all 32 lanes on each);
        // N = 128: lanes 0..15 take lines 0 and 2, lanes 16..31 lines 1 and 3.
        const int l0 = (CPL == 32) ? 0 : sub, l1 = (CPL == 32) ? 1 : 2 + sub;
        double s = scal[SC_S];
        double dtG = dt * (scal[SC_G] * scal[SC_S2]), dtD = dt * scal[SC_D];   // u = dt V + dtG |q|^2 + dtD Phi
        for (int i = warp; i < nmine; i += NW) {
            const int st = i % NST;
            // trap potential of this lane's two lines, V_y + V_z, and (batch) the member's scalars: global loads
            // issued before the wait for the tile, consumed after the transform
            const int row = (int)(tile_of(i) * LPT);
            const double vr0 = dt * (vy[(row + l0) % ny] + vz[((row + l0) / ny) % nz]);
            const double vr1 = dt * (vy[(row + l1) % ny] + vz[((row + l1) / ny) % nz]);
            if (nb > 1) {
                const double* sc = scal + (size_t)(row / (ny * nz)) * SC_COUNT;
                s = sc[SC_S]; dtG = dt * (sc[SC_G] * sc[SC_S2]); dtD = dt * sc[SC_D];
            }
            wait_issued(issued, i);
            mbar_wait(full + st, (i / NST) & 1);
            cd* ps = (cd*)(base + (size_t)st * PSI_BYTES);
            cd* slot = (cd*)(slots + (size_t)st * SLOT_BYTES);
            cd* sa = slot + pr * PAIR_EL;
            // ---- inverse transform of the pair's spectrum: v[j] = (Phi on line a, Phi on line b) at x = j*T + m
            {
                const cd* sb = sa + NXHP;
                cd v[P::V];
#pragma unroll
                for (int j = 0; j < P::V; ++j) {
                    const int k = j * T + m;
                    if (k <= N / 2) {
                        const cd a = sa[k], b = sb[k];
                        v[j] = cmake(a.x - b.y, a.y + b.x);          // X_a + i X_b
                    } else {
                        const cd a = sa[N - k], b = sb[N - k];
                        v[j] = cmake(a.x + b.y, b.x - a.y);          // conj X_a + i conj X_b
                    }
                }
                __syncwarp();                                        // the rows are in registers: reuse their area
                fftv_line_warp<P, +1>(v, m, sa, twA, tw2);
                __syncwarp();
                // (Phi on line a, Phi on line b) at x, one padded row of pairs: a lane's 8 consecutive x sit 144
                // bytes after its neighbour's
#pragma unroll
                for (int j = 0; j < P::V; ++j) sa[padt(j * T + m)] = v[j];
            }
            __syncwarp();
            // ---- calcnu on 8 consecutive points of two lines (registers u0, u1), then calclux on the same registers
            cd u0[WL], u1[WL];
            cd* p0 = ps + l0 * N + c * WL;                           // chunk c = 128-byte row c of the line, swizzled
            cd* p1 = ps + l1 * N + c * WL;
            const int sw = c & 7;
#pragma unroll
            for (int k = 0; k < WL; ++k) { u0[k] = p0[k ^ sw]; u1[k] = p1[k ^ sw]; }
            {
                // N = 256: both lines belong to pair 0, line 0 takes Phi.x and line 1 Phi.y of the same entries;
                // N = 128: slot s belongs to pair s, and `sub` says which component is this lane's line
                const cd* ph0 = slot + (l0 >> 1) * PAIR_EL + padt(c * WL);
                const cd* ph1 = slot + (l1 >> 1) * PAIR_EL + padt(c * WL);
                const double* vxc = vxs + padd(c * WL);
#pragma unroll
                for (int half = 0; half < 2; ++half) {
#pragma unroll
                    for (int k0 = 0; k0 < WL; k0 += NLW_C) {
                        cd* u = half ? u1 : u0;
                        const cd* ph = half ? ph1 : ph0;
                        const double vr = half ? vr1 : vr0;
                        const bool second = half ? (l1 & 1) : (l0 & 1);
                        double a[NLW_C];
#pragma unroll
                        for (int kk = 0; kk < NLW_C; ++kk) {
                            const cd f = ph[k0 + kk];
                            a[kk] = fma(dtD, second ? f.y : f.x, vxc[k0 + kk] + vr);
                            a[kk] = fma(dtG, cnorm2(u[k0 + kk]), a[kk]);
                        }
#pragma unroll
                        for (int kk = 0; kk < NLW_C; ++kk) {
                            if (RT) {
                                double sn, cs_;
                                sincos_cw(a[kk], &sn, &cs_);          // branch-free: the evaluations interleave
                                u[k0 + kk] = cmul(u[k0 + kk], cmake(cs_, -sn));      // (s = 1 in real time: no calcnorm, dbec_normalize applies its factor at once)
                            } else {
                                u[k0 + kk] = cmul(s * exp_cw(-a[kk]), u[k0 + kk]);
                            }
                        }
                    }
                }
            }
            // ---- calclux: neighbours by shuffle, zero-start recurrences, carries by shuffle (K terms)
            const cd zero = cmake(0.0, 0.0);
            cd lo0 = shfl_up_cd(u0[WL - 1], 1, CPL), hi0 = shfl_down_cd(u0[0], 1, CPL);
            cd lo1 = shfl_up_cd(u1[WL - 1], 1, CPL), hi1 = shfl_down_cd(u1[0], 1, CPL);
            if (c == 0) { lo0 = zero; lo1 = zero; }
            if (c == CPL - 1) { hi0 = zero; hi1 = zero; }
            const CT* hc = th + padt(c * WL);
            cn_chunk_forward2<CT>(u0, u1, lo0, hi0, lo1, hi1, kap, hc);
            cd d0 = zero, d1 = zero;
            for (int q = K; q >= 1; --q) {                           // D_in = e[c-1] + pfe[c-1] (e[c-2] + pfe[c-2] (...))
                const cd e0 = shfl_up_cd(u0[WL - 1], q, CPL), e1 = shfl_up_cd(u1[WL - 1], q, CPL);
                if (c - q >= 0) { const CT f = pfe[c - q]; d0 = cn_fma(f, d0, e0); d1 = cn_fma(f, d1, e1); }
            }
            const CT* pfc = tpf + padt(c * WL);
            cn_chunk_backward2<CT>(u0, u1, d0, d1, hc, pfc);
            cd w0 = zero, w1 = zero;
            for (int q = K; q >= 1; --q) {                           // U_in = e[c+1] + pbs[c+1] (e[c+2] + ...)
                const cd e0 = shfl_down_cd(u0[0], q, CPL), e1 = shfl_down_cd(u1[0], q, CPL);
                if (c + q < CPL) { const CT f = pbs[c + q]; w0 = cn_fma(f, w0, e0); w1 = cn_fma(f, w1, e1); }
            }
            const CT* pbc = tpb + padt(c * WL);
            cn_chunk_fix2<CT>(u0, u1, w0, w1, pbc);
#pragma unroll
            for (int k = 0; k < WL; ++k) { p0[k ^ sw] = u0[k]; p1[k ^ sw] = u1[k]; }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(done + st);
        }
    } else if (tid == NW * 32) {
        const uint64_t pol = l2_policy_code(pol_spec), polp = l2_policy_code(pol_ld);
        unsigned long long t0 = 0;
        for (int i = 0; i < nmine; ++i) {
            const int st = i % NST;
            if (i >= NST) mbar_wait(empty + st, ((i / NST) - 1) & 1);
            if (pace.ns) pace_wait(t0, i, pace);
            st_release_shared(issued, i + 1);
            mbar_expect_tx(full + st, PSI_BYTES + PAIRS * 2 * NXHP * (int)sizeof(cd));
            const long long tile = tile_of(i);
            tma_load_3d_hint(base + (size_t)st * PSI_BYTES, &map_psi, 0, 0, (int)(tile * LPT), full + st, polp);
#pragma unroll 1
            for (int pp = 0; pp < PAIRS; ++pp)
                bulk_load_hint(slots + (size_t)st * SLOT_BYTES + (size_t)pp * PAIR_EL * sizeof(cd),
                               spec + (tile * PAIRS + pp) * 2 * NXHP, 2 * NXHP * (int)sizeof(cd), full + st, pol);
        }
        if (pace.ns) pace_done(pace.st);
    } else if (tid == (NW + 1) * 32 || tid == (NW + 2) * 32) {
        // two storers (even / odd stages): while one sits in wait_group.read, the other drains the next stage
        const int which = warp - NW - 1;
        const uint64_t polp = l2_policy_code(pol_st);
        for (int i = 0; i < nmine; ++i) {
            const int st = i % NST;
            if ((st & 1) != which) continue;
            mbar_wait(done + st, (i / NST) & 1);
            tma_store_3d_hint(&map_psi, 0, 0, (int)(tile_of(i) * LPT), base + (size_t)st * PSI_BYTES, polp);
            bulk_commit();
            bulk_wait_read<0>();
            mbar_arrive(empty + st);
        }
        bulk_wait<0>();
    }
}

// ------------------------------------------------------------------------------------------------
// lines of 512 points: TWO warps per line pair
// ------------------------------------------------------------------------------------------------
// A pair of 512-point lines is 16 KiB of psi plus 9 KiB of spectrum / exchange: with one warp per pair only seven
// warps' worth of stages fit.  Here the two warps of a group share the pair: the 64 threads run the pair's inverse
// transform together (V = 8, T = 64: the exchanges are 64-thread named barriers), then each warp takes ONE line:
// a lane holds chunks `lane` and `lane + 32` of it (8 points each), calcnu and calclux as in k_xwarp_nonlin, the
// neighbours, chunk ends and carries crossing between the two halves by rotating shuffles.
typedef FftPlanV<8, 8, 8> WPlan512;

__device__ __forceinline__ cd shfl_rot_cd(cd v, int src) {
    return cmake(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}

template <bool RT, int NG, int NST>
__global__ void __launch_bounds__((2 * NG + 3) * 32, 1)
k_xwarp2_nonlin(const __grid_constant__ CUtensorMap map_psi, const cd* __restrict__ spec, const cd* __restrict__ twN_g,
                const double* __restrict__ scal, const double* __restrict__ vx_g, const double* __restrict__ vy,
                const double* __restrict__ vz, double dt, int ntiles, int ny, int nz, int nb, CnTabW<RT> cn, int rev,
                float pol_ld, float pol_st, float pol_spec, PaceArgs pace) {
    typedef typename CnCoef<RT>::type CT;
    typedef WPlan512 P;
    constexpr int N = 512, NLW_C = RT ? 2 : NlwBatch<RT>::C;
    constexpr int T = P::T;                                          // 64 threads per pair
    constexpr int CPL = N / WL;                                      // 64 chunks per line: two per lane
    constexpr int NXHP = w_nxhp(N);
    constexpr int NTAB = N + N / 8;
    constexpr int PAIR_EL = w_pair_el(P::SMEM, NXHP, NTAB);
    constexpr int NPD = N + N / 4;
    constexpr int PSI_BYTES = 2 * N * (int)sizeof(cd), SLOT_BYTES = PAIR_EL * (int)sizeof(cd);
    static_assert(PSI_BYTES % 1024 == 0, "the swizzle pattern needs 1024-byte aligned psi tiles");
    constexpr int NW = 2 * NG, NT = (NW + 3) * 32;
    extern __shared__ __align__(1024) unsigned char smraw[];
    unsigned char* base = smraw;
    unsigned char* slots = base + (size_t)NST * PSI_BYTES;
    cd* tw = (cd*)(slots + (size_t)NST * SLOT_BYTES);            // twA [N], tw2 [T]
    CT* tab = (CT*)(tw + N + T);                                 // h, PF, PB (padded), PFE, PBS
    double* vxs = (double*)(tab + 3 * NTAB + 2 * CPL);
    uint64_t* bars = (uint64_t*)(vxs + NPD);
    uint64_t* full = bars; uint64_t* empty = bars + NST; uint64_t* done = bars + 2 * NST;
    int* issued = (int*)(bars + 3 * NST);
    const int tid = threadIdx.x;
    for (int k = tid; k < N; k += NT) {
        tw[k] = twN_g[((k % T) * (k / T)) % N];                  // twA[k1*T + m] = W_N^{m k1}
        if (k < T) tw[N + k] = twN_g[(P::V * (k % P::R3) * (k / P::R3)) % N];   // tw2[k2*R3 + n3] = W_N^{V n3 k2}
        vxs[padd(k)] = dt * vx_g[k];
        tab[padt(k)] = cn.h[k]; tab[NTAB + padt(k)] = cn.pf[k]; tab[2 * NTAB + padt(k)] = cn.pb[k];
    }
    for (int k = tid; k < CPL; k += NT) { tab[3 * NTAB + k] = cn.pfe[k]; tab[3 * NTAB + CPL + k] = cn.pbs[k]; }
    if (tid == 0) {
        *issued = 0;
        for (int s = 0; s < NST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); mbar_init(done + s, 2); }
        fence_mbar_init();
    }
    __syncthreads();
    pdl_launch_dependents();
    pdl_wait();
    const int nmine = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    auto tile_of = [&](int i) {
        const long long t = (long long)blockIdx.x + (long long)i * gridDim.x;
        return rev ? (long long)ntiles - 1 - t : t;
    };
    const int warp = tid >> 5, lane = tid & 31;
    if (warp < NW) {
        const cd* twA = tw; const cd* tw2 = tw + N;
        const CT* th = tab; const CT* tpf = tab + NTAB; const CT* tpb = tab + 2 * NTAB;
        const CT* pfe = tab + 3 * NTAB; const CT* pbs = pfe + CPL;
        const CT kap = cn.kap;
        const int K = cn.K;
        const int g = warp >> 1, sub = warp & 1;                     // group, and this warp's line of the pair
        const int m = tid - g * 64;                                  // FFT thread of the pair
        const int c0 = lane, c1 = lane + 32;                         // this lane's two chunks of the line
        double s = scal[SC_S];
        double dtG = dt * (scal[SC_G] * scal[SC_S2]), dtD = dt * scal[SC_D];
        for (int i = g; i < nmine; i += NG) {
            const int st = i % NST;
            const int row = (int)(tile_of(i) * 2) + sub;
            const double vr = dt * (vy[row % ny] + vz[(row / ny) % nz]);
            if (nb > 1) {
                const double* sc = scal + (size_t)(row / (ny * nz)) * SC_COUNT;
                s = sc[SC_S]; dtG = dt * (sc[SC_G] * sc[SC_S2]); dtD = dt * sc[SC_D];
            }
            wait_issued(issued, i);
            mbar_wait(full + st, (i / NST) & 1);
            cd* ps = (cd*)(base + (size_t)st * PSI_BYTES);
            cd* sa = (cd*)(slots + (size_t)st * SLOT_BYTES);
            // ---- inverse transform of the pair's spectrum by the group's 64 threads
            {
                const cd* sb = sa + NXHP;
                cd v[P::V];
#pragma unroll
                for (int j = 0; j < P::V; ++j) {
                    const int k = j * T + m;
                    if (k <= N / 2) {
                        const cd a = sa[k], b = sb[k];
                        v[j] = cmake(a.x - b.y, a.y + b.x);          // X_a + i X_b
                    } else {
                        const cd a = sa[N - k], b = sb[N - k];
                        v[j] = cmake(a.x + b.y, b.x - a.y);          // conj X_a + i conj X_b
                    }
                }
                named_bar_sync(1 + g, 64);                           // the rows are in registers: reuse their area
                fftv_stage1<P, +1>(v, m, twA);
                fftv_x1_write<P>(v, m, sa);
                named_bar_sync(1 + g, 64);
                fftv_stage2<P, +1>(v, m, sa, tw2);
                named_bar_sync(1 + g, 64);
                fftv_x2_write<P>(v, m, sa);
                named_bar_sync(1 + g, 64);
                fftv_stage3<P, +1>(v, m, sa);
                named_bar_sync(1 + g, 64);
#pragma unroll
                for (int j = 0; j < P::V; ++j) sa[padt(j * T + m)] = v[j];       // (Phi line a, Phi line b) at x
            }
            named_bar_sync(1 + g, 64);
            // ---- calcnu on this warp's line: chunks c0 and c1 in registers u0, u1
            cd u0[WL], u1[WL];
            cd* p0 = ps + sub * N + c0 * WL;
            cd* p1 = ps + sub * N + c1 * WL;
            const int sw = lane & 7;                                 // (c0 & 7 == c1 & 7)
#pragma unroll
            for (int k = 0; k < WL; ++k) { u0[k] = p0[k ^ sw]; u1[k] = p1[k ^ sw]; }
            {
                const cd* ph0 = sa + padt(c0 * WL);
                const cd* ph1 = sa + padt(c1 * WL);
                const double* vx0 = vxs + padd(c0 * WL);
                const double* vx1 = vxs + padd(c1 * WL);
#pragma unroll
                for (int half = 0; half < 2; ++half) {
#pragma unroll
                    for (int k0 = 0; k0 < WL; k0 += NLW_C) {
                        cd* u = half ? u1 : u0;
                        const cd* ph = half ? ph1 : ph0;
                        const double* vxc = half ? vx1 : vx0;
                        double a[NLW_C];
#pragma unroll
                        for (int kk = 0; kk < NLW_C; ++kk) {
                            const cd f = ph[k0 + kk];
                            a[kk] = fma(dtD, sub ? f.y : f.x, vxc[k0 + kk] + vr);
                            a[kk] = fma(dtG, cnorm2(u[k0 + kk]), a[kk]);
                        }
#pragma unroll
                        for (int kk = 0; kk < NLW_C; ++kk) {
                            if (RT) {
                                double sn, cs_;
                                sincos_cw(a[kk], &sn, &cs_);
                                u[k0 + kk] = cmul(u[k0 + kk], cmake(cs_, -sn));      // (s = 1 in real time: no calcnorm, dbec_normalize applies its factor at once)
                            } else {
                                u[k0 + kk] = cmul(s * exp_cw(-a[kk]), u[k0 + kk]);
                            }
                        }
                    }
                }
            }
            // ---- calclux on 64 chunks: chunk lane (u0) and chunk lane + 32 (u1)
            const cd zero = cmake(0.0, 0.0);
            const int up = (lane + 31) & 31, dn = (lane + 1) & 31;
            {
                const cd a = shfl_rot_cd(u0[WL - 1], up), b = shfl_rot_cd(u1[WL - 1], up);
                const cd c = shfl_rot_cd(u1[0], dn), d = shfl_rot_cd(u0[0], dn);
                const cd lo0 = lane > 0 ? a : zero, lo1 = lane > 0 ? b : a;      // chunk 32 follows chunk 31 (lane 31's u0)
                const cd hi0 = lane < 31 ? d : c, hi1 = lane < 31 ? c : zero;    // chunk 31 precedes chunk 32 (lane 0's u1)
                cn_chunk_forward<CT>(u0, lo0, hi0, kap, th + padt(c0 * WL));
                cn_chunk_forward<CT>(u1, lo1, hi1, kap, th + padt(c1 * WL));
            }
            cd d0 = zero, d1 = zero;
            for (int q = K; q >= 1; --q) {                           // D_in = e[c-1] + pfe[c-1] (e[c-2] + pfe[c-2] (...))
                const int src = (lane - q) & 31;
                const cd r0 = shfl_rot_cd(u0[WL - 1], src), r1 = shfl_rot_cd(u1[WL - 1], src);
                if (lane >= q) d0 = cn_fma(pfe[c0 - q], d0, r0);
                d1 = cn_fma(pfe[c1 - q], d1, lane >= q ? r1 : r0);
            }
            cn_chunk_backward<CT>(u0, d0, th + padt(c0 * WL), tpf + padt(c0 * WL));
            cn_chunk_backward<CT>(u1, d1, th + padt(c1 * WL), tpf + padt(c1 * WL));
            cd w0 = zero, w1 = zero;
            for (int q = K; q >= 1; --q) {                           // U_in = e[c+1] + pbs[c+1] (e[c+2] + ...)
                const int src = (lane + q) & 31;
                const cd r0 = shfl_rot_cd(u0[0], src), r1 = shfl_rot_cd(u1[0], src);
                w0 = cn_fma(pbs[c0 + q], w0, lane + q < 32 ? r0 : r1);
                if (lane + q < 32) w1 = cn_fma(pbs[c1 + q], w1, r1);
            }
            cn_chunk_fix<CT>(u0, w0, tpb + padt(c0 * WL));
            cn_chunk_fix<CT>(u1, w1, tpb + padt(c1 * WL));
#pragma unroll
            for (int k = 0; k < WL; ++k) { p0[k ^ sw] = u0[k]; p1[k ^ sw] = u1[k]; }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(done + st);
        }
    } else if (tid == NW * 32) {
        const uint64_t pol = l2_policy_code(pol_spec), polp = l2_policy_code(pol_ld);
        unsigned long long t0 = 0;
        for (int i = 0; i < nmine; ++i) {
            const int st = i % NST;
            if (i >= NST) mbar_wait(empty + st, ((i / NST) - 1) & 1);
            if (pace.ns) pace_wait(t0, i, pace);
            st_release_shared(issued, i + 1);
            mbar_expect_tx(full + st, PSI_BYTES + 2 * NXHP * (int)sizeof(cd));
            const long long tile = tile_of(i);
            tma_load_3d_hint(base + (size_t)st * PSI_BYTES, &map_psi, 0, 0, (int)(tile * 2), full + st, polp);
            bulk_load_hint(slots + (size_t)st * SLOT_BYTES, spec + tile * 2 * NXHP, 2 * NXHP * (int)sizeof(cd), full + st, pol);
        }
        if (pace.ns) pace_done(pace.st);
    } else if (tid == (NW + 1) * 32 || tid == (NW + 2) * 32) {
        const int which = warp - NW - 1;
        const uint64_t polp = l2_policy_code(pol_st);
        for (int i = 0; i < nmine; ++i) {
            const int st = i % NST;
            if ((st & 1) != which) continue;
            mbar_wait(done + st, (i / NST) & 1);
            tma_store_3d_hint(&map_psi, 0, 0, (int)(tile_of(i) * 2), base + (size_t)st * PSI_BYTES, polp);
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
// These kernels are bound by the fp64 pipe, not by memory: paced to the slowest CTA (tma_pipe.cuh: pace_wait) they lose
// 8 - 30 % (measured at 256^3 and 512 x 512 x 256); the loaders keep the hook, the launchers switch it off.
static PaceArgs no_pace() { PaceArgs pa; pa.ns = 0; pa.head = 0; pa.head_ns = 0; pa.st = nullptr; return pa; }

template <bool RT> static CnTabW<RT> make_cntabw(const AxisTables& a);
template <> CnTabW<true> make_cntabw<true>(const AxisTables& a) {
    CnTabW<true> t; t.h = a.h; t.pf = a.pf8; t.pb = a.pb8; t.pfe = a.pfe8; t.pbs = a.pbs8; t.kap = a.kap; t.K = a.K8; return t;
}
template <> CnTabW<false> make_cntabw<false>(const AxisTables& a) {
    CnTabW<false> t; t.h = a.h_re; t.pf = a.pf8_re; t.pb = a.pb8_re; t.pfe = a.pfe8_re; t.pbs = a.pbs8_re; t.kap = a.kap.x; t.K = a.K8;
    return t;
}

int dbec_xwarp_supported(const dbec_handle_s* h) {
    const int lpt = h->nx == 128 ? 4 : 2;
    // 512-point lines: the two-warps-per-pair kernel stages 45 KB of tables per CTA before its first tile; a grid
    // with only a tile or two per SM (BASELINE.json's 512^2 config: 256 pairs) is served faster by k_xline_nonlin
    if (h->nx == 512 && (long long)h->ny * h->nplanes / 2 < 8LL * h->num_sms) return 0;
    return h->use_tma && h->fuse_cnx && (h->nx == 128 || h->nx == 256 || h->nx == 512) && ((h->ny * h->nz) % lpt == 0) &&
           h->ax[0].K8 >= 1 && h->ax[0].K8 <= 31;
}

template <int N, bool RT, int NW, int NST> static int launch_xwarp(dbec_handle_s* h) {
    typedef typename CnCoef<RT>::type CT;
    typedef typename WPlan<N>::P P;
    constexpr int PAIRS = 32 / P::T, LPT = 2 * PAIRS, NXHP = w_nxhp(N), CPL = N / WL;
    constexpr int PAIR_EL = w_pair_el(P::SMEM, NXHP, N + N / 8);
    constexpr int STAGE = LPT * N * (int)sizeof(cd) + PAIRS * PAIR_EL * (int)sizeof(cd);
    if (h->nxhp != NXHP) return (int)cudaErrorInvalidValue;
    const int ntiles = (int)((long long)h->ny * h->nplanes / LPT);
    const int grid = ntiles < h->num_sms ? ntiles : h->num_sms;
    const size_t sm = (size_t)NST * STAGE + (N + P::T) * sizeof(cd) + (3 * (N + N / 8) + 2 * CPL) * sizeof(CT) +
                      (N + N / 4) * sizeof(double) + (3 * NST + 1) * sizeof(uint64_t);
    auto k = k_xwarp_nonlin<N, RT, NW, NST>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const CUtensorMap* map = (const CUtensorMap*)h->tmap[TM_PSI_XW];
    CK(launch_pdl(k, dim3(grid), dim3((NW + 3) * 32), sm, h->stream, h->use_pdl, *map, (const cd*)h->spec, h->ax[0].twN,
                  (const double*)h->scal, h->ax[0].vtrap, h->ax[1].vtrap, h->ax[2].vtrap, h->p.dt, ntiles, h->ny, h->nz, h->nb,
                  make_cntabw<RT>(h->ax[0]), h->rev_next, h->pol[POL_NL_LD], h->pol[POL_NL_ST], h->pol[POL_NL_SPEC], no_pace()));
    h->launches++;
    return (int)cudaGetLastError();
}

template <bool RT, int NG, int NST> static int launch_xwarp2(dbec_handle_s* h) {
    typedef typename CnCoef<RT>::type CT;
    typedef WPlan512 P;
    constexpr int N = 512, NXHP = w_nxhp(N), CPL = N / WL;
    constexpr int PAIR_EL = w_pair_el(P::SMEM, NXHP, N + N / 8);
    constexpr int STAGE = 2 * N * (int)sizeof(cd) + PAIR_EL * (int)sizeof(cd);
    if (h->nxhp != NXHP) return (int)cudaErrorInvalidValue;
    const int ntiles = (int)((long long)h->ny * h->nplanes / 2);
    const int grid = ntiles < h->num_sms ? ntiles : h->num_sms;
    const size_t sm = (size_t)NST * STAGE + (N + P::T) * sizeof(cd) + (3 * (N + N / 8) + 2 * CPL) * sizeof(CT) +
                      (N + N / 4) * sizeof(double) + (3 * NST + 1) * sizeof(uint64_t);
    auto k = k_xwarp2_nonlin<RT, NG, NST>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const CUtensorMap* map = (const CUtensorMap*)h->tmap[TM_PSI_XW];
    CK(launch_pdl(k, dim3(grid), dim3((2 * NG + 3) * 32), sm, h->stream, h->use_pdl, *map, (const cd*)h->spec, h->ax[0].twN,
                  (const double*)h->scal, h->ax[0].vtrap, h->ax[1].vtrap, h->ax[2].vtrap, h->p.dt, ntiles, h->ny, h->nz, h->nb,
                  make_cntabw<RT>(h->ax[0]), h->rev_next, h->pol[POL_NL_LD], h->pol[POL_NL_ST], h->pol[POL_NL_SPEC], no_pace()));
    h->launches++;
    return (int)cudaGetLastError();
}

int dbec_launch_xwarp_nonlin(dbec_handle_s* h) {
    const bool rt = h->p.time_mode == 1;
    switch (h->nx) {
        case 512: return rt ? launch_xwarp2<true, 6, 7>(h) : launch_xwarp2<false, 6, 7>(h);
        case 128: return rt ? launch_xwarp<128, true, 12, 15>(h) : launch_xwarp<128, false, 12, 15>(h);
        case 256: return rt ? launch_xwarp<256, true, 12, 16>(h) : launch_xwarp<256, false, 12, 16>(h);
        default: return (int)cudaErrorInvalidValue;
    }
}
