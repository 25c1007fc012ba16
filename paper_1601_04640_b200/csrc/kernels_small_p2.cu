// kernels_small_p2.cu — the one-launch cluster step (kernels_small.cu) for small 3-D grids whose three lengths are
// powers of two known at compile time (16, 32 or 64 each, up to 128 Ki points: BASELINE.json's 32^3 config).  Same passes A - D, same data flow through L2,
// same cluster barriers; what changes is how a line is worked on.  k_small_step serves any length, so its transforms
// are Stockham passes through shared memory with a block barrier after each (about 40 per step, 900 cycles per
// pass) and its code does not fit the instruction cache.  Here a line of N points belongs to N/4 lanes of ONE warp:
//   * transforms in registers (fft_linev.cuh, 4 values per lane), exchanges through a per-warp scratch with
//     __syncwarp; forward, V_dd multiply and inverse of pass B never leave the registers;
//   * the split / merge of the two-real-lines transform happens while loading the next transform;
//   * Crank-Nicolson sweeps on chunks of 8 points, N/8 lanes per line, neighbours and carries by warp shuffles;
//   * global loads and stores go straight from / to the registers of the lane that needs them.
// Five block barriers (two more for the norm in imaginary time) and four cluster barriers per step.  Results agree with k_small_step to round-off (another
// summation order in the transforms); tests/test_gpu_parity.py runs both against the oracle.
//
// Cubes (NY == NZ) need only THREE cluster barriers per step: the roles of y and z alternate from step to step.
// An even step works as described (planes of fixed z in A and C, lines along z in B and D) and ends with every
// CTA holding, after its calcluz, all x and z for its own rows of y; the odd step that follows starts right
// there, without a barrier: its "planes" are those of fixed y (A: density, FFT-x, FFT-z; C: inverse FFT-z,
// inverse FFT-x, calcnu, calclux, calcluz) and its lines run along y (B: FFT-y, x V_dd, inverse; D: calcluy), which
// leaves every CTA with the planes of fixed z the next even step begins on.  The transforms of the three axes
// are applied in another order and calcluy / calcluz swap places — the sweeps act on different indices and
// commute exactly (pinned for the oracle by tests/test_oracle_pins.py), so the difference is round-off.  In
// imaginary time the norm factor is then read one barrier later (after pass A, whose density is linear in it:
// pass B multiplies by s^2 instead).
#include <cooperative_groups.h>
#include "dbec_internal.hpp"
#include "fft_linev.cuh"
#include "cn_chunk.cuh"
#include "cn_line_smem.cuh"
#include "trig.cuh"

namespace cg = cooperative_groups;

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return (int)e_; } while (0)

constexpr int P2T = 512;            // threads per CTA
constexpr int P2L = 8;              // points per Crank-Nicolson chunk

template <int N> struct P2Plan;
template <> struct P2Plan<16> { typedef FftPlanV<4, 4, 1> P; };
template <> struct P2Plan<32> { typedef FftPlanV<4, 4, 2> P; };
template <> struct P2Plan<64> { typedef FftPlanV<4, 4, 4> P; };

struct P2Args {
    cd* psi; cd* spec; const double* vdd; double* scal;
    const cd* tw[3];                // exp(-2 pi i j / n) per axis
    const double* vt[3];            // trap potential per axis
    int nb, nsteps, imag, nyf, nxhp;
    double dt, dV;
    long long P, SP;
};

__host__ __device__ constexpr int p2_skew(int k) { return k + (k >> 3); }       // one pad element per 8 entries
__device__ __forceinline__ cd p2_ldcg(const cd* p) { return __ldcg(p); }      // L2 only: other SMs rewrite these lines
__device__ __forceinline__ cd p2_shfl(cd a, int src) {
    return cmake(__shfl_sync(0xffffffffu, a.x, src), __shfl_sync(0xffffffffu, a.y, src));
}

// Twiddle tables of a plan from the axis table tw[j] = exp(-2 pi i j / N):
// twA[k1 T + m] = W^(m k1), tw2[k2 R3 + n3] = W^(V n3 k2)   (fft_linev.cuh)
template <class P> __device__ __forceinline__ void p2_make_tw(const cd* __restrict__ tw, cd* twA, cd* tw2) {
    for (int i = threadIdx.x; i < P::N; i += P2T) { const int k1 = i / P::T, m = i % P::T; twA[i] = tw[(m * k1) % P::N]; }
    for (int i = threadIdx.x; i < P::T; i += P2T) { const int k2 = i / P::R3, n3 = i % P::R3; tw2[i] = tw[(P::V * n3 * k2) % P::N]; }
}

// Crank-Nicolson solve (cn_chunk.cuh) of one line held by NCH lanes of a warp, 8 points each; c = this lane's chunk.
// Neighbour points and chunk carries travel by shuffles (lane of chunk i = l0 + i ls).  All 32 lanes must call.
template <bool RT, int NCH>
__device__ __forceinline__ void p2_cn(cd (&u)[P2L], int c, int l0, int ls, const typename CnCoef<RT>::type* h,
                                      const typename CnCoef<RT>::type* pf, const typename CnCoef<RT>::type* pb,
                                      const typename CnCoef<RT>::type* pfe, const typename CnCoef<RT>::type* pbs,
                                      typename CnCoef<RT>::type kap) {
    typedef typename CnCoef<RT>::type CT;
    const cd zero = cmake(0.0, 0.0);
    cd lo = p2_shfl(u[P2L - 1], l0 + (c > 0 ? c - 1 : 0) * ls);
    cd hi = p2_shfl(u[0], l0 + (c < NCH - 1 ? c + 1 : c) * ls);
    if (c == 0) lo = zero;
    if (c == NCH - 1) hi = zero;
    cn_chunk_forward<CT>(u, lo, hi, kap, h + c * (P2L + 1));
    const cd e = u[P2L - 1];
    cd din = zero;
#pragma unroll
    for (int i = 0; i < NCH - 1; ++i) {
        const cd ei = p2_shfl(e, l0 + i * ls);
        if (i < c) din = cn_fma(pfe[i], din, ei);
    }
    cn_chunk_backward<CT>(u, din, h + c * (P2L + 1), pf + c * (P2L + 1));
    const cd e1 = u[0];
    cd uin = zero;
#pragma unroll
    for (int i = NCH - 1; i > 0; --i) {
        const cd ei = p2_shfl(e1, l0 + i * ls);
        if (i > c) uin = cn_fma(pbs[i], uin, ei);
    }
    cn_chunk_fix<CT>(u, uin, pb + c * (P2L + 1));
}

// Sum over the block in a fixed order; every thread receives the result.
__device__ __forceinline__ double p2_block_sum_all(double x, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) red[w] = x;
    __syncthreads();
    double t = 0.0;
    for (int i = 0; i < P2T / 32; ++i) t += red[i];
    return t;
}

// Shared-memory layout (elements of cd unless noted), the same on host and device.
// Planes of a CTA's slab that passes A and C hold in shared memory at a time: all NZ / CS of them if they fit, else
// the largest power-of-two part that does (a small cluster then walks its slab in several rounds).
__host__ __device__ constexpr int p2_pps(int nx, int ny, int nz, int cs) {
    int pps = nz / cs;
    while (pps > 1 && (pps % 2 == 0) &&
           (size_t)(pps * ny) * ((nx + nx / 8 + 3) / 8 * 8 + 4 + nx / 2 + nx / 2 + 1) * sizeof(cd) > 170 * 1024) pps /= 2;
    return pps;
}

template <bool RT, int NX, int NY, int NZ, int CS> struct P2Lay {
    static_assert(NZ % CS == 0 && (NZ / CS * NY) % 2 == 0, "whole planes and whole pairs of rows per CTA");
    typedef typename P2Plan<NX>::P PX; typedef typename P2Plan<NY>::P PY; typedef typename P2Plan<NZ>::P PZ;
    static constexpr int PPC = NZ / CS;                 // planes per CTA
    static constexpr int PPS = p2_pps(NX, NY, NZ, CS);  // ... of which passes A and C work on at a time
    static_assert(PPC % PPS == 0 && (PPS * NY) % 2 == 0, "whole rounds, whole pairs of rows");
    static constexpr int R = PPS * NY, NP = R / 2;        // rows / pairs of rows of one round
    static constexpr int NXH1 = NX / 2 + 1;               // half-spectrum length
    // a psi row in shared memory: point x at x + x/8 (p2_skew: the chunks of a row start in different bank groups),
    // row pitch = 4 mod 8 (two neighbouring rows complement each other)
    static constexpr int PP = (NX + NX / 8 + 3) / 8 * 8 + 4;
    static constexpr int cmax(int a, int b) { return a > b ? a : b; }
    static constexpr int up8(int a) { return (a + 7) / 8 * 8; }
    // exchange scratch of one line; the pitch between the lines of a warp keeps the 8 lanes of a quarter warp in 8
    // different 16-byte bank groups: contiguous lanes (x) — lines of fewer than 8 lanes sit T groups apart; interleaved
    // lanes (y, z: 32/T lines side by side) — T/4 groups apart
    static constexpr int SX = up8(PX::SMEM) + (PX::T < 8 ? PX::T : 0), SY = up8(PY::SMEM) + PY::T / 4, SZ = up8(PZ::SMEM) + PZ::T / 4;
    static constexpr int SCRW = cmax(cmax((32 / PX::T) * SX, (32 / PY::T) * SY), (32 / PZ::T) * SZ);
    static constexpr int o_pb = 0, o_zb = o_pb + R * PP, o_xb = o_zb + NP * NX, o_scr = o_xb + R * NXH1;
    static constexpr int o_tw = o_scr + (P2T / 32) * SCRW;                       // twA, tw2 of x, y, z
    static constexpr int n_tw = NX + PX::T + NY + PY::T + NZ + PZ::T;
    static constexpr int o_cn = o_tw + n_tw;                                     // per axis: h, pf, pb (N), pfe, pbs (N/8), as CT
    static constexpr int n_cn = 3 * (NX + NY + NZ) * 9 / 8 + 2 * (NX + NY + NZ) / P2L;   // counted as complex in either time mode
    static constexpr int o_v = o_cn + n_cn;                                      // trap tables, doubles
    static constexpr int total = o_v + (NX + NY + NZ + 1) / 2 + 1;
    static constexpr size_t bytes = (size_t)total * sizeof(cd);
};

template <bool RT, int NX, int NY, int NZ, int CS>
__global__ void __launch_bounds__(P2T, 1)
k_small_p2(const __grid_constant__ P2Args a, CnTab<RT> cnx_g, CnTab<RT> cny_g, CnTab<RT> cnz_g) {
    typedef P2Lay<RT, NX, NY, NZ, CS> LY;
    typedef typename LY::PX PX; typedef typename LY::PY PY; typedef typename LY::PZ PZ;
    typedef typename CnCoef<RT>::type CT;
    constexpr int R = LY::R, NP = LY::NP, NXH1 = LY::NXH1, PP = LY::PP, PPC = LY::PPC, PPS = LY::PPS, NSUB = PPC / PPS;
    constexpr int TX = PX::T, TY = PY::T, TZ = PZ::T, LPWY = 32 / TY, LPWZ = 32 / TZ;
    constexpr int NCHX = NX / P2L, NCHY = NY / P2L, NCHZ = NZ / P2L;
    extern __shared__ __align__(16) cd psm[];
    __shared__ double sc[SC_COUNT];             // this member's scalars (dbec_internal.hpp)
    __shared__ double red[P2T / 32];
    __shared__ double cpart;                    // this CTA's part of sum |psi|^2, read by the whole cluster
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int cid = (int)(blockIdx.x / CS), ncl = (int)(gridDim.x / CS);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    cd* Pb = psm + LY::o_pb; cd* ZB = psm + LY::o_zb; cd* XB = psm + LY::o_xb;
    cd* scr = psm + LY::o_scr + warp * LY::SCRW;
    cd* twAx = psm + LY::o_tw; cd* tw2x = twAx + NX; cd* twAy = tw2x + TX; cd* tw2y = twAy + NY; cd* twAz = tw2y + TY; cd* tw2z = twAz + NZ;
    // per axis: h, PF, PB (N entries), PF at chunk ends, PB at chunk starts (N/8): the 8-point chunk tables
    // (entry k of h, PF, PB at p2_skew(k): the chunks a warp works on start in different banks)
    constexpr int EX = NX + NCHX, EY = NY + NCHY, EZ = NZ + NCHZ;
    CT* tcx = (CT*)(psm + LY::o_cn); CT* tcy = tcx + 3 * EX + 2 * NCHX; CT* tcz = tcy + 3 * EY + 2 * NCHY;
    double* vxs = (double*)(psm + LY::o_v); double* vys = vxs + NX; double* vzs = vys + NY;
    // (staged once: a cluster barrier is an acquire and drops the L1 copies of global data, kernels_small.cu)
    p2_make_tw<PX>(a.tw[0], twAx, tw2x);
    p2_make_tw<PY>(a.tw[1], twAy, tw2y);
    p2_make_tw<PZ>(a.tw[2], twAz, tw2z);
    for (int k = tid; k < NX; k += P2T) { const int q = p2_skew(k); tcx[q] = cnx_g.h[k]; tcx[EX + q] = cnx_g.pf[k]; tcx[2 * EX + q] = cnx_g.pb[k]; vxs[k] = a.vt[0][k]; }
    for (int k = tid; k < NY; k += P2T) { const int q = p2_skew(k); tcy[q] = cny_g.h[k]; tcy[EY + q] = cny_g.pf[k]; tcy[2 * EY + q] = cny_g.pb[k]; vys[k] = a.vt[1][k]; }
    for (int k = tid; k < NZ; k += P2T) { const int q = p2_skew(k); tcz[q] = cnz_g.h[k]; tcz[EZ + q] = cnz_g.pf[k]; tcz[2 * EZ + q] = cnz_g.pb[k]; vzs[k] = a.vt[2][k]; }
    for (int k = tid; k < NCHX; k += P2T) { tcx[3 * EX + k] = cnx_g.pfe[k]; tcx[3 * EX + NCHX + k] = cnx_g.pbs[k]; }
    for (int k = tid; k < NCHY; k += P2T) { tcy[3 * EY + k] = cny_g.pfe[k]; tcy[3 * EY + NCHY + k] = cny_g.pbs[k]; }
    for (int k = tid; k < NCHZ; k += P2T) { tcz[3 * EZ + k] = cnz_g.pfe[k]; tcz[3 * EZ + NCHZ + k] = cnz_g.pbs[k]; }
    const int nxhp = a.nxhp;
    const size_t ls_spec = (size_t)NY * nxhp, vls = (size_t)a.nyf * nxhp;
    constexpr int QS = NY * NXH1, qs = (QS + CS - 1) / CS, QP = NY * NX, qp = (QP + CS - 1) / CS;
    const int qs_lo = min(QS, rank * qs), ncs = min(QS, qs_lo + qs) - qs_lo;      // last-axis columns of the spectrum
    const int qp_lo = min(QP, rank * qp), ncp = min(QP, qp_lo + qp) - qp_lo;      // ... of psi
    const cd zero = cmake(0.0, 0.0);
    constexpr bool SWAP = NY == NZ;           // y and z may trade places (header comment)

    for (int mem = cid; mem < a.nb; mem += ncl) {
        cd* psi = a.psi + (size_t)mem * a.P;
        cd* spec = a.spec + (size_t)mem * a.SP;
        double* scal = a.scal + (size_t)mem * SC_COUNT;
        __syncthreads();
        if (tid < SC_COUNT) sc[tid] = scal[tid];
        __syncthreads();
        bool pending = false;           // imaginary time: the CTAs' parts of the last norm wait in cpart
        for (int step = 0; step < a.nsteps; ++step) {
            if (tid == 0) ramp_advance(sc);                      // reading S26 (G, D are used in pass C)
            // this step's geometry: sw = y and z trade places.  Element strides of psi / spec: from plane to plane
            // of this CTA's slab (psP, spP) and from row to row inside a plane (psQ, spQ); the lines of passes B
            // and D run along the slab direction.  V_dd table: vQ per row, vL along the line.
            const bool sw = SWAP && (step & 1);
            const int psP = sw ? NX : NY * NX, psQ = sw ? NY * NX : NX;
            const size_t spP = sw ? (size_t)nxhp : ls_spec, spQ = sw ? ls_spec : (size_t)nxhp;
            const size_t vQ = sw ? vls : (size_t)nxhp, vL = sw ? (size_t)nxhp : vls;
            const CT* tq = sw ? tcz : tcy; const CT* tl = sw ? tcy : tcz;       // Crank-Nicolson tables: in-plane, line
            const CT kq = sw ? cnz_g.kap : cny_g.kap, kl = sw ? cny_g.kap : cnz_g.kap;
            const double* vq = sw ? vzs : vys; const double* vp = sw ? vys : vzs;
            // ---------------- A: density -> FFT-x -> split -> FFT-y -> spectrum ----------------
            for (int ss = 0; ss < NSUB; ++ss) {
                const int pl0 = rank * PPC + ss * PPS;                  // first plane of this round
                // (|psi|^2 without the norm factor: pass B multiplies by s^2)
                for (int base = 0; base < NP * TX; base += P2T) {
                    const int item = base + tid, line = item / TX, m = item % TX;
                    const bool act = line < NP;
                    const int r = act ? 2 * line : 0;
                    const cd* g = psi + (size_t)(pl0 + r / NY) * psP + (size_t)(r % NY) * psQ;
                    cd v[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        v[j] = zero;
                        if (act) {
                            const cd p0 = p2_ldcg(g + j * TX + m), p1 = p2_ldcg(g + psQ + j * TX + m);
                            v[j] = cmake(cnorm2(p0), cnorm2(p1));
                        }
                    }
                    __syncwarp();
                    fftv_line_warp<PX, -1>(v, m, scr + (lane / TX) * LY::SX, twAx, tw2x);
                    if (act) {
#pragma unroll
                        for (int j = 0; j < 4; ++j) ZB[line * NX + j * TX + m] = v[j];
                    }
                }
            __syncthreads();
            for (int base = 0; base < (PPS * NXH1 + LPWY - 1) / LPWY * 32; base += P2T) {
                const int line = ((base + tid) >> 5) * LPWY + lane % LPWY, m = lane / LPWY;
                const bool act = line < PPS * NXH1;
                const int p = act ? line / NXH1 : 0, k = act ? line % NXH1 : 0;
                cd v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    // X_a = (Z[k] + conj Z[N-k])/2 (even row),  X_b = (Z[k] - conj Z[N-k])/(2i) (odd row)
                    const int row = p * NY + j * TY + m, l = row >> 1;
                    const cd zk = ZB[l * NX + k], zp = ZB[l * NX + (k ? NX - k : 0)];
                    v[j] = (row & 1) ? cmake(0.5 * (zk.y + zp.y), -0.5 * (zk.x - zp.x)) : cmake(0.5 * (zk.x + zp.x), 0.5 * (zk.y - zp.y));
                }
                __syncwarp();
                fftv_line_warp<PY, -1>(v, m, scr + (lane % LPWY) * LY::SY, twAy, tw2y);
                if (act) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) spec[(size_t)(pl0 + p) * spP + (size_t)(j * TY + m) * spQ + k] = v[j];
                }
            }
            if (NSUB > 1) __syncthreads();              // the next round overwrites ZB
            }
            cluster.sync();
            if (pending) {
                // calcnorm of the previous step (reading S13): the CTAs' partial sums in rank order, the
                // same in every CTA
                if (tid == 0) {
                    double tot = 0.0;
                    for (int r = 0; r < CS; ++r) tot += *cluster.map_shared_rank(&cpart, r);
                    const double sf = 1.0 / sqrt(tot * a.dV);
                    sc[SC_S] = sf; sc[SC_S2] = sf * sf;
                }
                __syncthreads();
                pending = false;
            }
            // ---------------- B: FFT-z, x V_dd(k)/P, inverse FFT-z, all in registers ----------------
            for (int base = 0; base < (ncs + LPWZ - 1) / LPWZ * 32; base += P2T) {
                const int col = ((base + tid) >> 5) * LPWZ + lane % LPWZ, m = lane / LPWZ;
                const bool act = col < ncs;
                const int q = qs_lo + (act ? col : 0), y = q / NXH1, k = q % NXH1;
                cd* gc = spec + (size_t)y * spQ + k;
                // folded table (dbec_internal.hpp): index m and N - m share an entry
                const double* vd = a.vdd + (size_t)(y < NY - y ? y : NY - y) * vQ + k;
                const double s2 = sc[SC_S2];
                cd v[4];
                double w[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int z = j * TZ + m;
                    v[j] = act ? p2_ldcg(gc + z * spP) : zero;
                    w[j] = act ? s2 * __ldg(vd + (size_t)(z < NZ - z ? z : NZ - z) * vL) : 0.0;
                }
                __syncwarp();
                fftv_line_warp<PZ, -1>(v, m, scr + (lane % LPWZ) * LY::SZ, twAz, tw2z);
#pragma unroll
                for (int j = 0; j < 4; ++j) v[j] = cmul(w[j], v[j]);
                __syncwarp();
                fftv_line_warp<PZ, +1>(v, m, scr + (lane % LPWZ) * LY::SZ, twAz, tw2z);
                if (act) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) gc[(j * TZ + m) * spP] = v[j];
                }
            }
            // psi of this CTA's rows for the first round of pass C: pass B does not touch psi, so the loads fly
            // while the cluster barrier and the inverse y transforms run
            cd q0[4], q1[4];
            if (NSUB == 1) {
                const int line = tid / TX, m = tid % TX, r = line < NP ? 2 * line : 0;
                const cd* g0 = psi + (size_t)(rank * PPC + r / NY) * psP + (size_t)(r % NY) * psQ;
#pragma unroll
                for (int j = 0; j < 4; ++j) { q0[j] = p2_ldcg(g0 + j * TX + m); q1[j] = p2_ldcg(g0 + psQ + j * TX + m); }
            }
            cluster.sync();
            // ---------------- C: inverse FFT-y -> merge -> inverse FFT-x -> calcnu -> calclux -> calcluy ----------------
            for (int ss = 0; ss < NSUB; ++ss) {
            const int pl0 = rank * PPC + ss * PPS;                      // first plane of this round
            for (int base = 0; base < (PPS * NXH1 + LPWY - 1) / LPWY * 32; base += P2T) {
                const int line = ((base + tid) >> 5) * LPWY + lane % LPWY, m = lane / LPWY;
                const bool act = line < PPS * NXH1;
                const int p = act ? line / NXH1 : 0, k = act ? line % NXH1 : 0;
                cd v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) v[j] = act ? p2_ldcg(spec + (size_t)(pl0 + p) * spP + (size_t)(j * TY + m) * spQ + k) : zero;
                __syncwarp();
                fftv_line_warp<PY, +1>(v, m, scr + (lane % LPWY) * LY::SY, twAy, tw2y);
                if (act) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) XB[(p * NY + j * TY + m) * NXH1 + k] = v[j];
                }
            }
            __syncthreads();
            {
                const double s = sc[SC_S], s2 = sc[SC_S2], G = sc[SC_G], D = sc[SC_D], dt = a.dt;
                for (int base = 0; base < NP * TX; base += P2T) {
                    const int item = base + tid, line = item / TX, m = item % TX;
                    const bool act = line < NP;
                    const int l = act ? line : 0;
                    const cd* ra = XB + (2 * l) * NXH1;
                    const cd* rb = ra + NXH1;
                    const cd* g0 = psi + (size_t)(pl0 + (2 * l) / NY) * psP + (size_t)((2 * l) % NY) * psQ;
                    cd v[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int kk = j * TX + m;
                        if (NSUB > 1 || base > 0) { q0[j] = p2_ldcg(g0 + kk); q1[j] = p2_ldcg(g0 + psQ + kk); }
                        // X_a + i X_b on 0 .. N/2, the conjugates above
                        if (kk <= NX / 2) { const cd p = ra[kk], q = rb[kk]; v[j] = cmake(p.x - q.y, p.y + q.x); }
                        else { const cd p = ra[NX - kk], q = rb[NX - kk]; v[j] = cmake(p.x + q.y, q.x - p.y); }
                    }
                    __syncwarp();
                    fftv_line_warp<PX, +1>(v, m, scr + (lane / TX) * LY::SX, twAx, tw2x);     // (Phi row 2l, Phi row 2l+1)
                    if (act) {
#pragma unroll
                        for (int hr = 0; hr < 2; ++hr) {
                            const int row = 2 * l + hr, y = row % NY, zz = pl0 + row / NY;
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const int x = j * TX + m;
                                const cd q = hr ? q1[j] : q0[j];
                                const double u = dt * (vxs[x] + vq[y] + vp[zz] + G * (s2 * cnorm2(q)) + D * (hr ? v[j].y : v[j].x));
                                cd w;
                                if (RT) { double sn, cs; sincos_cw(u, &sn, &cs); w = cmul(s, cmul(q, cmake(cs, -sn))); }
                                else w = cmul(s * exp_cw(-u), q);
                                Pb[row * PP + p2_skew(x)] = w;
                            }
                        }
                    }
                }
            }
            __syncthreads();
            for (int base = 0; base < R * NCHX; base += P2T) {                    // calclux: a row = NCHX neighbouring lanes
                const int item = base + tid, c = item % NCHX;
                const bool act = item < R * NCHX;
                cd* g = Pb + (act ? item / NCHX : 0) * PP + c * (P2L + 1);
                cd u[P2L];
#pragma unroll
                for (int i = 0; i < P2L; ++i) u[i] = g[i];
                p2_cn<RT, NCHX>(u, c, lane - c, 1, tcx, tcx + EX, tcx + 2 * EX, tcx + 3 * EX, tcx + 3 * EX + NCHX, cnx_g.kap);
                if (act) {
#pragma unroll
                    for (int i = 0; i < P2L; ++i) g[i] = u[i];
                }
            }
            __syncthreads();
            {
                constexpr int LPW = 32 / NCHY;                                    // calcluy: lane = chunk LPW + column
                for (int base = 0; base < (PPS * NX + LPW - 1) / LPW * 32; base += P2T) {
                    const int col = ((base + tid) >> 5) * LPW + lane % LPW, c = lane / LPW;
                    const bool act = col < PPS * NX;
                    const int p = act ? col / NX : 0, x = act ? col % NX : 0;
                    cd* g = Pb + (p * NY + c * P2L) * PP + p2_skew(x);
                    cd u[P2L];
#pragma unroll
                    for (int i = 0; i < P2L; ++i) u[i] = g[i * PP];
                    p2_cn<RT, NCHY>(u, c, lane % LPW, LPW, tq, tq + EY, tq + 2 * EY, tq + 3 * EY, tq + 3 * EY + NCHY, kq);
                    if (act) {
                        // straight to global memory: the LPW neighbouring columns of a chunk are one contiguous piece
                        cd* go = psi + (size_t)(pl0 + p) * psP + (size_t)(c * P2L) * psQ + x;
#pragma unroll
                        for (int i = 0; i < P2L; ++i) go[(size_t)i * psQ] = u[i];
                    }
                }
            }
            if (NSUB > 1) __syncthreads();              // the next round overwrites XB and Pb
            }
            cluster.sync();
            // ---------------- D: calcluz from / to global memory (+ calcnorm) ----------------
            double acc = 0.0;
            {
                constexpr int LPW = 32 / NCHZ;
                for (int base = 0; base < (ncp + LPW - 1) / LPW * 32; base += P2T) {
                    const int col = ((base + tid) >> 5) * LPW + lane % LPW, c = lane / LPW;
                    const bool act = col < ncp;
                    const int qq = qp_lo + (act ? col : 0);
                    cd* g = psi + (size_t)(c * P2L) * psP + (size_t)(qq / NX) * psQ + qq % NX;
                    cd u[P2L];
#pragma unroll
                    for (int i = 0; i < P2L; ++i) u[i] = act ? p2_ldcg(g + i * psP) : zero;
                    p2_cn<RT, NCHZ>(u, c, lane % LPW, LPW, tl, tl + EZ, tl + 2 * EZ, tl + 3 * EZ, tl + 3 * EZ + NCHZ, kl);
                    if (act) {
#pragma unroll
                        for (int i = 0; i < P2L; ++i) { g[i * psP] = u[i]; acc += cnorm2(u[i]); }
                    }
                }
            }
            if (a.imag) {
                const double part = p2_block_sum_all(acc, red);
                if (tid == 0) cpart = part;
                pending = true;             // read after the next cluster barrier
            }
            // a cube's next step starts on what this CTA has just written (header comment): block barrier only
            if (SWAP) __syncthreads(); else cluster.sync();
        }
        if (pending) {
            cluster.sync();
            if (tid == 0) {
                double tot = 0.0;
                for (int r = 0; r < CS; ++r) tot += *cluster.map_shared_rank(&cpart, r);
                const double sf = 1.0 / sqrt(tot * a.dV);
                sc[SC_S] = sf; sc[SC_S2] = sf * sf;
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
// chunk tables of 8 points as a CnTab (cn_line_smem.cuh holds the 16-point ones)
template <bool RT> static CnTab<RT> p2_cntab8(const AxisTables& a);
template <> CnTab<true> p2_cntab8<true>(const AxisTables& a) {
    CnTab<true> t; t.h = a.h; t.pf = a.pf8; t.pb = a.pb8; t.pfe = a.pfe8; t.pbs = a.pbs8; t.kap = a.kap; t.K = a.K8; return t;
}
template <> CnTab<false> p2_cntab8<false>(const AxisTables& a) {
    CnTab<false> t; t.h = a.h_re; t.pf = a.pf8_re; t.pb = a.pb8_re; t.pfe = a.pfe8_re; t.pbs = a.pbs8_re; t.kap = a.kap.x; t.K = a.K8;
    return t;
}

static void p2_config(cudaLaunchConfig_t* cfg, cudaLaunchAttribute* at, size_t smem, int cs, int nclusters, cudaStream_t st) {
    *cfg = cudaLaunchConfig_t();
    cfg->gridDim = dim3(cs * nclusters); cfg->blockDim = dim3(P2T); cfg->dynamicSmemBytes = smem; cfg->stream = st;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg->attrs = at; cfg->numAttrs = 1;
}

// what = 0: clusters of this instantiation that can be resident at once (0: cannot run); what = 1: launch nsteps steps
template <bool RT, int NX, int NY, int NZ, int CS> static int p2_run(dbec_handle_s* h, int what, int nsteps) {
    auto k = k_small_p2<RT, NX, NY, NZ, CS>;
    const size_t smem = P2Lay<RT, NX, NY, NZ, CS>::bytes;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    if (what == 0) {
        if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
            cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) { cudaGetLastError(); return 0; }
        p2_config(&cfg, at, smem, CS, 1, h->stream);
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, k, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
        return n;
    }
    P2Args a;
    a.psi = h->psi; a.spec = h->spec; a.vdd = h->vdd; a.scal = h->scal;
    for (int ax = 0; ax < 3; ++ax) { a.tw[ax] = h->ax[ax].twN; a.vt[ax] = h->ax[ax].vtrap; }
    a.nb = h->nb; a.nsteps = nsteps; a.imag = h->p.time_mode == 0; a.nyf = h->nyf; a.nxhp = h->nxhp;
    a.dt = h->p.dt; a.dV = h->dV; a.P = h->P; a.SP = h->SP;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    p2_config(&cfg, at, smem, CS, h->nb < h->small_max_clusters ? h->nb : h->small_max_clusters, h->stream);
    CK(cudaLaunchKernelEx(&cfg, k, a, p2_cntab8<RT>(h->ax[0]), p2_cntab8<RT>(h->ax[1]), p2_cntab8<RT>(h->ax[2])));
    h->launches++;
    return (int)cudaGetLastError();
}

// the shapes and cluster sizes this file is compiled for (NX, NY, NZ, CTAs per cluster): every grid of up to 128 Ki
// points whose lengths are 16, 32 or 64, on 16 CTAs (64^3 is left to the multi-launch path: 62 us per step there,
// 97 here); the cubes also on smaller clusters, which give a member fewer SMs and a batch more members in flight
#define P2_SHAPES(X) X(16, 16, 16, 16) X(16, 16, 32, 16) X(16, 16, 64, 16) X(16, 32, 16, 16) X(16, 32, 32, 16) \
                     X(16, 32, 64, 16) X(16, 64, 16, 16) X(16, 64, 32, 16) X(16, 64, 64, 16) X(32, 16, 16, 16) \
                     X(32, 16, 32, 16) X(32, 16, 64, 16) X(32, 32, 16, 16) X(32, 32, 32, 16) X(32, 32, 64, 16) \
                     X(32, 64, 16, 16) X(32, 64, 32, 16) X(64, 16, 16, 16) X(64, 16, 32, 16) X(64, 16, 64, 16) \
                     X(64, 32, 16, 16) X(64, 32, 32, 16) X(64, 64, 16, 16) X(16, 16, 16, 4) X(16, 16, 16, 1) \
                     X(32, 32, 32, 8) X(32, 32, 32, 4) X(32, 32, 32, 2) \
                     X(64, 64, 32, 16) X(32, 64, 64, 16) X(64, 32, 64, 16)
static const int p2_cluster_sizes[] = {16, 8, 4, 2, 1};

static int p2_dispatch(dbec_handle_s* h, int cs, int what, int nsteps) {
    const bool rt = h->p.time_mode == 1;
#define P2_CASE(NX, NY, NZ, CS) \
    if (h->nx == NX && h->ny == NY && h->nz == NZ && cs == CS) \
        return rt ? p2_run<true, NX, NY, NZ, CS>(h, what, nsteps) : p2_run<false, NX, NY, NZ, CS>(h, what, nsteps);
    P2_SHAPES(P2_CASE)
#undef P2_CASE
    return what == 0 ? 0 : (int)cudaErrorInvalidValue;
}

// CTAs per cluster (and h->small_max_clusters set) when dbec_step of this handle can run in k_small_p2 — a 3-D grid
// of one of the compiled shapes with the 8-point chunk tables built — else 0.  request > 0: that cluster size or
// nothing.  Otherwise the choice is by the time one step of the whole batch takes: a cluster works through
// ceil(nb / resident clusters) members one after the other, and a member's step costs about 9 us + 4.1 ns per grid
// point of a CTA's share (measured on B200 — 16^3: 10.7 us on 16 CTAs, 11.5 on 4, 20.6 on 1; 32^3: 16.2 us on 16,
// 23.1 on 8, 41.0 on 4, 76.0 on 2).  So one 32^3 grid takes 16 CTAs, 64 of them take clusters of 2 (76.8 us per
// batch step against 161 on 16 CTAs, of which 8 are resident, and 151 through the seven launches), 256 grids of 16^3
// single CTAs (41 us against 149).
static double p2_step_cost(const dbec_handle_s* h, int cs) { return 9.0 + 0.0041 * (double)h->P / cs; }

int dbec_small_p2_choose(dbec_handle_s* h, int request) {
    if (h->p.ndim != 3 || h->ax[0].K8 < 1 || h->ax[1].K8 < 1 || h->ax[2].K8 < 1) return 0;
    int best = 0, best_n = 0;
    double best_t = 0.0;
    for (int cs : p2_cluster_sizes) {
        if (request > 0 && cs != request) continue;
        const int n = p2_dispatch(h, cs, 0, 0);
        if (n < 1) continue;
        const double t = (double)((h->nb + n - 1) / n) * p2_step_cost(h, cs);
        if (!best || t < best_t) { best = cs; best_n = n; best_t = t; }
    }
    if (best) h->small_max_clusters = best_n;
    return best;
}

int dbec_launch_small_p2(dbec_handle_s* h, int nsteps) { return p2_dispatch(h, h->use_cluster, 1, nsteps); }
