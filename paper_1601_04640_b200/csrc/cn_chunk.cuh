// cn_chunk.cuh — chunked Crank-Nicolson (Thomas) recurrences for one grid line.
//
// calclux / calcluy / calcluz ("recursive relation"): on each line solve
//   -a u_{j-1} + (1+2a) u_j - a u_{j+1} = a p_{j-1} + (1-2a) p_j + a p_{j+1},  u_0 = u_{N-1} = 0,
// a = c dt / (4 h^2), c = 1 (imaginary time) or i (real time)  [reading S11].
//
// Thomas elimination with the constant off-diagonal folded into one table h_j = a / den_j,
// den_1 = 1+2a, den_j = 1+2a - a h_{j-1}, and h_0 = h_{N-1} = 0 (Dirichlet ends):
//   forward   d_j = h_j (r'_j + d_{j-1}),   r'_j = p_{j-1} + p_{j+1} + kap p_j,  kap = (1-2a)/a
//   backward  u_j = d_j + h_j u_{j+1}
// The paper runs one thread over the whole line.  Here a line is cut into chunks of
// CN_L points, one thread per chunk, all chunks of a line advancing at once: each chunk runs the
// recurrence from a zero start, the true incoming value D_in reaches element j through the
// precomputable product PF_j = h_{j0} ... h_j  (d_j = d~_j + PF_j D_in), and D_in itself is a short
// Horner recurrence over the chunk ends.  Same for the backward pass with PB_j = h_j ... h_{jend}.
// This is the scan the paper set aside for its launch count done inside one kernel.
#pragma once
#include "cplx.cuh"

#define CN_L 16

// coefficient type: real in imaginary time, complex in real time
template <bool RT> struct CnCoef { typedef double type; };
template <> struct CnCoef<true> { typedef cd type; };

DBEC_HD cd cn_mul(double h, cd a) { return cmul(h, a); }
DBEC_HD cd cn_mul(cd h, cd a) { return cmul(h, a); }
DBEC_HD cd cn_fma(double h, cd a, cd b) { return cfma(h, a, b); }   // b + h*a
DBEC_HD cd cn_fma(cd h, cd a, cd b) { return cfma(h, a, b); }

// Forward pass on one chunk from a zero start.  u[i] = p_{j0+i} on entry, d~_{j0+i} on exit.
// lo = p_{j0-1}, hi = p_{j0+L} (0 outside the line).  h points at h_{j0}.
// (The chunk length L is deduced from the register array: 16 in the tile kernels, 8 in the warp-per-line kernel.)
template <class CT, int L> DBEC_HD void cn_chunk_forward(cd (&u)[L], cd lo, cd hi, CT kap, const CT* __restrict__ h) {
    cd prev = lo, d = cmake(0.0, 0.0);
#pragma unroll
    for (int i = 0; i < L; ++i) {
        cd cur = u[i];
        cd nxt = (i + 1 < L) ? u[i + 1] : hi;
        cd r = cn_fma(kap, cur, cadd(prev, nxt));
        d = cn_mul(h[i], cadd(r, d));
        u[i] = d;
        prev = cur;
    }
}

// Backward pass on one chunk: applies the forward fix-up (d_j = d~_j + PF_j D_in) and runs
// u~_j = d_j + h_j u~_{j+1} from a zero start.  u[i] = u~_{j0+i} on exit.
template <class CT, int L> DBEC_HD void cn_chunk_backward(cd (&u)[L], cd d_in, const CT* __restrict__ h,
                                                          const CT* __restrict__ pf) {
    cd ut = cmake(0.0, 0.0);
#pragma unroll
    for (int i = L - 1; i >= 0; --i) {
        cd dj = cn_fma(pf[i], d_in, u[i]);
        ut = cn_fma(h[i], ut, dj);
        u[i] = ut;
    }
}

// Final fix-up: u_j = u~_j + PB_j U_in.
template <class CT, int L> DBEC_HD void cn_chunk_fix(cd (&u)[L], cd u_in, const CT* __restrict__ pb) {
#pragma unroll
    for (int i = 0; i < L; ++i) u[i] = cn_fma(pb[i], u_in, u[i]);
}

// The same three steps on the chunks of TWO lines at once (same chunk position, same tables): every table
// entry is loaded once for both, and the two dependent chains interleave.
template <class CT, int L> DBEC_HD void cn_chunk_forward2(cd (&u)[L], cd (&w)[L], cd lou, cd hiu, cd low, cd hiw, CT kap,
                                                          const CT* __restrict__ h) {
    cd pu = lou, pw = low, du = cmake(0.0, 0.0), dw = cmake(0.0, 0.0);
#pragma unroll
    for (int i = 0; i < L; ++i) {
        const CT hh = h[i];
        const cd cu = u[i], cw = w[i];
        const cd nu = (i + 1 < L) ? u[i + 1] : hiu, nw = (i + 1 < L) ? w[i + 1] : hiw;
        du = cn_mul(hh, cadd(cn_fma(kap, cu, cadd(pu, nu)), du));
        dw = cn_mul(hh, cadd(cn_fma(kap, cw, cadd(pw, nw)), dw));
        u[i] = du; w[i] = dw;
        pu = cu; pw = cw;
    }
}
template <class CT, int L> DBEC_HD void cn_chunk_backward2(cd (&u)[L], cd (&w)[L], cd du_in, cd dw_in, const CT* __restrict__ h,
                                                           const CT* __restrict__ pf) {
    cd tu = cmake(0.0, 0.0), tw = cmake(0.0, 0.0);
#pragma unroll
    for (int i = L - 1; i >= 0; --i) {
        const CT hh = h[i], pp = pf[i];
        tu = cn_fma(hh, tu, cn_fma(pp, du_in, u[i]));
        tw = cn_fma(hh, tw, cn_fma(pp, dw_in, w[i]));
        u[i] = tu; w[i] = tw;
    }
}
template <class CT, int L> DBEC_HD void cn_chunk_fix2(cd (&u)[L], cd (&w)[L], cd uu_in, cd uw_in, const CT* __restrict__ pb) {
#pragma unroll
    for (int i = 0; i < L; ++i) {
        const CT pp = pb[i];
        u[i] = cn_fma(pp, uu_in, u[i]);
        w[i] = cn_fma(pp, uw_in, w[i]);
    }
}

// Carry into chunk c of the forward pass: D_in = d_{c*L-1}, from the zero-start chunk ends
// e[i*es] = d~ at the last element of chunk i and pfend[i] = PF at that element.
// K: the number of terms that are above 2^-73 of the first (the factors are products of CN_L consecutive |h_j| < 1;
// dbec_api.cu carry_terms) — the sum starts K chunks back; the default takes them all.
template <class CT> DBEC_HD cd cn_carry_forward(int c, const cd* e, int es, const CT* __restrict__ pfend, int K = 1 << 30) {
    cd D = cmake(0.0, 0.0);
    for (int i = (c - K > 0 ? c - K : 0); i < c; ++i) D = cn_fma(pfend[i], D, e[i * es]);
    return D;
}

// Carry into chunk c of the backward pass: U_in = u_{(c+1)*L}, from chunk starts
// e[i*es] = u~ at the first element of chunk i and pbstart[i] = PB at that element.
template <class CT> DBEC_HD cd cn_carry_backward(int c, int C, const cd* e, int es, const CT* __restrict__ pbstart, int K = 1 << 30) {
    cd U = cmake(0.0, 0.0);
    for (int i = (K < C - 1 - c ? c + K : C - 1); i > c; --i) U = cn_fma(pbstart[i], U, e[i * es]);
    return U;
}
