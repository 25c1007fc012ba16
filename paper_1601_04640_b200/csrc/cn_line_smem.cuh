// cn_line_smem.cuh — Crank-Nicolson solve (calclux) of one contiguous grid line
// that the T = N/16 threads of a warp hold in the strided register layout of the line FFT
// (q[j] = line[j*T + m]).  The line is transposed through a padded shared-memory row into chunks
// of 16 consecutive points per thread (cn_chunk.cuh), solved, and transposed back.
#pragma once
#include "dbec_internal.hpp"
#include "cn_chunk.cuh"

template <bool RT> struct CnTab {
    typedef typename CnCoef<RT>::type CT;
    const CT* h; const CT* pf; const CT* pb; const CT* pfe; const CT* pbs;
    CT kap;
    int K;              // carry terms above 2^-73 of the first one (AxisTables::K16)
};
template <bool RT> inline CnTab<RT> make_cntab(const AxisTables& a);
template <> inline CnTab<true> make_cntab<true>(const AxisTables& a) {
    CnTab<true> t; t.h = a.h; t.pf = a.pf; t.pb = a.pb; t.pfe = a.pfe; t.pbs = a.pbs; t.kap = a.kap; t.K = a.K16; return t;
}
template <> inline CnTab<false> make_cntab<false>(const AxisTables& a) {
    CnTab<false> t; t.h = a.h_re; t.pf = a.pf_re; t.pb = a.pb_re; t.pfe = a.pfe_re; t.pbs = a.pbs_re; t.kap = a.kap.x; t.K = a.K16;
    return t;
}

// Shared row of N + 3T elements: point k at k + (k >> 4) (one pad element per chunk keeps the
// chunked reads conflict-free), then T forward chunk ends and T backward chunk starts.
// TS: distance between the table entries of consecutive chunks (16 for the plain global tables, 17
// for tables staged in shared memory with one pad element per chunk, see cn_stage_tables).
template <bool RT, int T, int TS>
__device__ __forceinline__ void cn_line_via_smem(cd (&q)[16], int m, cd* sm, const CnTab<RT>& cn) {
    typedef typename CnCoef<RT>::type CT;
    constexpr int N = 16 * T;
#pragma unroll
    for (int j = 0; j < 16; ++j) { const int k = j * T + m; sm[k + (k >> 4)] = q[j]; }
    __syncwarp();
    const int j0 = 16 * m;
    cd u[CN_L];
#pragma unroll
    for (int i = 0; i < CN_L; ++i) u[i] = sm[j0 + m + i];
    const cd lo = (m > 0) ? sm[j0 - 1 + (m - 1)] : cmake(0.0, 0.0);
    const cd hi = (m < T - 1) ? sm[j0 + 16 + m + 1] : cmake(0.0, 0.0);
    cd* ends = sm + N + T;
    cn_chunk_forward<CT>(u, lo, hi, cn.kap, cn.h + TS * m);
    ends[m] = u[CN_L - 1];
    __syncwarp();
    const cd din = cn_carry_forward<CT>(m, ends, 1, cn.pfe);
    cn_chunk_backward<CT>(u, din, cn.h + TS * m, cn.pf + TS * m);
    ends[T + m] = u[0];
    __syncwarp();
    const cd uin = cn_carry_backward<CT>(m, T, ends + T, 1, cn.pbs);
    cn_chunk_fix<CT>(u, uin, cn.pb + TS * m);
#pragma unroll
    for (int i = 0; i < CN_L; ++i) sm[j0 + m + i] = u[i];
    __syncwarp();
#pragma unroll
    for (int j = 0; j < 16; ++j) { const int k = j * T + m; q[j] = sm[k + (k >> 4)]; }
}

// Stage the h / PF / PB tables of an axis in shared memory, entry k at k + (k >> 4): the 16 chunks a
// warp works on then hit 16 different bank groups (straight from global memory the same reads are
// 16 separate 128-byte lines per load instruction).  Returns the table set pointing at the copies.
// Needs 3 * cn_tab_elems(N) elements of CT at `buf`; the caller synchronises the block afterwards.
__host__ __device__ constexpr int cn_tab_elems(int n) { return (n + n / 16 + 1) & ~1; }
template <bool RT, int N>
__device__ __forceinline__ CnTab<RT> cn_stage_tables(const CnTab<RT>& g, typename CnCoef<RT>::type* buf) {
    constexpr int E = cn_tab_elems(N);
    for (int k = threadIdx.x; k < N; k += blockDim.x) {
        const int p = k + (k >> 4);
        buf[p] = g.h[k];
        buf[E + p] = g.pf[k];
        buf[2 * E + p] = g.pb[k];
    }
    CnTab<RT> t = g;
    t.h = buf; t.pf = buf + E; t.pb = buf + 2 * E;
    return t;
}
