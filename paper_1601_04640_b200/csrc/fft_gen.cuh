// fft_gen.cuh — run-time-length line FFT in shared memory: a Stockham autosort transform, one radix-r pass
// (r = 4, 2, 3, 5, 7) per factor of N, twiddles from the axis' table exp(-2 pi i j / N).  The DFT of PAPER.md:63
// for line lengths N = 2^a 3^b 5^c 7^d that the register-resident plans of fft_line.cuh do not cover
// (kernels_gen.cu) and for the cluster-resident small-grid step (kernels_small.cu).
// Product path only; nothing here is used by oracle/.
#pragma once
#include "fft_line.cuh"

struct GenPlan {
    int n, nfac;
    int fac[12];        // radices in the order they are applied
};

// One radix-R Stockham butterfly.  in / out: element e of the line at e*SE.  Ns = product of the radices already
// applied, nb = n / R, j < nb.  twN[j] = exp(-2 pi i j / n); S = -1 forward, +1 inverse.
template <int R, int S>
__device__ __forceinline__ void gen_butterfly(const cd* in, cd* out, int SE, int j, int Ns, int nb, int n, const cd* __restrict__ twN) {
    const int k = j % Ns;
    cd v[R];
    const int tstep = (n / (Ns * R)) * k;                    // W_{Ns R}^{k t} = twN[t * tstep]
#pragma unroll
    for (int t = 0; t < R; ++t) {
        v[t] = in[(j + t * nb) * SE];
        if (t > 0) v[t] = cmul(v[t], tw_dir<S>(twN[t * tstep]));      // t * tstep < n
    }
    if (R == 2) dft2<S>(v[0], v[1]);
    else if (R == 4) dft4<S>(v[0], v[1], v[2], v[3]);
    else {                                                   // 3, 5, 7: the definition, roots W_R^q = twN[q n / R]
        cd w[R];
#pragma unroll
        for (int q = 0; q < R; ++q) {
            cd acc = v[0];
#pragma unroll
            for (int t = 1; t < R; ++t) acc = cfma(v[t], tw_dir<S>(twN[((q * t) % R) * (n / R)]), acc);
            w[q] = acc;
        }
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = w[q];
    }
    const int j0 = (j - k) * R + k;
#pragma unroll
    for (int t = 0; t < R; ++t) out[(j0 + t * Ns) * SE] = v[t];
}

// Transform L lines held in shared memory (line l starts at l*SL, element stride SE) with all threads of the
// block; a and b are the two Stockham buffers.  LFAST: the line index runs fastest over the threads (tiles of
// neighbouring columns) or the butterfly index does (contiguous lines).  Returns the buffer holding the result.
template <int S, bool LFAST>
__device__ __forceinline__ cd* gen_fft_lines(cd* a, cd* b, int L, int SL, int SE, const GenPlan& pl, const cd* __restrict__ twN) {
    int Ns = 1;
    for (int s = 0; s < pl.nfac; ++s) {
        const int r = pl.fac[s], nb = pl.n / r;
        for (int idx = threadIdx.x; idx < L * nb; idx += blockDim.x) {
            const int l = LFAST ? idx % L : idx / nb, j = LFAST ? idx / L : idx % nb;
            const cd* in = a + l * SL;
            cd* out = b + l * SL;
            switch (r) {
                case 2: gen_butterfly<2, S>(in, out, SE, j, Ns, nb, pl.n, twN); break;
                case 3: gen_butterfly<3, S>(in, out, SE, j, Ns, nb, pl.n, twN); break;
                case 4: gen_butterfly<4, S>(in, out, SE, j, Ns, nb, pl.n, twN); break;
                case 5: gen_butterfly<5, S>(in, out, SE, j, Ns, nb, pl.n, twN); break;
                default: gen_butterfly<7, S>(in, out, SE, j, Ns, nb, pl.n, twN); break;
            }
        }
        __syncthreads();
        cd* t = a; a = b; b = t;
        Ns *= r;
    }
    return a;
}

// Division by a run-time constant as one multiply-high: exact while x * d < 2^32 (indices here stay below 2^17,
// divisors below 2^12).  m = 0 stands for d = 1.
struct FastDiv {
    unsigned d, m;
    __host__ __device__ FastDiv() : d(1), m(0) {}
    __host__ __device__ explicit FastDiv(int dd) : d((unsigned)dd), m(dd > 1 ? 0xFFFFFFFFu / (unsigned)dd + 1u : 0u) {}
#if defined(__CUDACC__)
    __device__ __forceinline__ int div(int x) const { return m ? (int)__umulhi((unsigned)x, m) : x; }
    __device__ __forceinline__ void divmod(int x, int& q, int& r) const { q = div(x); r = x - q * (int)d; }
#endif
};

// One radix-R Stockham butterfly with the index arithmetic done by the caller: k = j % Ns, tstep = (n / (Ns R)) k.
// FIRST: Ns = 1, all twiddles are 1.
template <int R, int S, bool FIRST>
__device__ __forceinline__ void gen_butterfly_k(const cd* in, cd* out, int SE, int j, int k, int Ns, int nb, int n, int tstep,
                                                const cd* __restrict__ twN) {
    cd v[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
        v[t] = in[(j + t * nb) * SE];
        if (!FIRST && t > 0) v[t] = cmul(v[t], tw_dir<S>(twN[t * tstep]));      // t * tstep < n
    }
    if (R == 2) dft2<S>(v[0], v[1]);
    else if (R == 4) dft4<S>(v[0], v[1], v[2], v[3]);
    else if (R == 8 || R == 16) dft_small<R, S>(v);
    else {
        cd w[R];
#pragma unroll
        for (int q = 0; q < R; ++q) {
            cd acc = v[0];
#pragma unroll
            for (int t = 1; t < R; ++t) acc = cfma(v[t], tw_dir<S>(twN[((q * t) % R) * nb]), acc);      // nb = n / R
            w[q] = acc;
        }
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = w[q];
    }
    const int j0 = (j - k) * R + k;
#pragma unroll
    for (int t = 0; t < R; ++t) out[(j0 + t * Ns) * SE] = v[t];
}

// A plan with everything a pass needs worked out on the host (no division on the device): radix r, butterflies per
// line nb = n / r, product of the earlier radices Ns, twiddle step n / (Ns r), and the multiply-high constants of
// nb and Ns.
struct GenPass { int r, nb, Ns, tunit; FastDiv fnb, fNs; };
struct GenPlanP { int n, nfac; GenPass pass[10]; };      // lengths up to 1024 have at most 6 radices (729 = 3^6)
inline bool make_plan_p(const GenPlan& g, GenPlanP* p) {
    p->n = g.n; p->nfac = g.nfac;
    if (g.nfac > 10) return false;
    int Ns = 1;
    for (int s = 0; s < g.nfac; ++s) {
        GenPass& q = p->pass[s];
        q.r = g.fac[s]; q.nb = g.n / q.r; q.Ns = Ns; q.tunit = g.n / (Ns * q.r);
        q.fnb = FastDiv(q.nb); q.fNs = FastDiv(Ns);
        Ns *= q.r;
    }
    for (int s = g.nfac; s < 10; ++s) { p->pass[s] = GenPass(); p->pass[s].r = 0; }
    return true;
}

// One pass of the transform below: L lines, nb butterflies each.
template <int R, int S, bool LFAST>
__device__ __forceinline__ void gen_fft_pass(const cd* a, cd* b, int L, const FastDiv& fL, const FastDiv& fL0, int S0, int S1, int SE,
                                             int n, const GenPass& ps, const cd* __restrict__ twN) {
    const int nb = ps.nb, Ns = ps.Ns, tunit = ps.tunit;
    const FastDiv fnb = ps.fnb, fNs = ps.fNs;
    for (int idx = threadIdx.x; idx < L * nb; idx += blockDim.x) {
        int l, j, lq, lr, jq, k;
        if (LFAST) fL.divmod(idx, j, l); else fnb.divmod(idx, l, j);
        fL0.divmod(l, lq, lr);
        const int off = lq * S1 + lr * S0;
        fNs.divmod(j, jq, k);
        gen_butterfly_k<R, S, false>(a + off, b + off, SE, j, k, Ns, nb, n, tunit * k, twN);
    }
}
// the odd radices are rare: one out-of-line copy each keeps the calling kernel inside the instruction cache
template <int R, int S, bool LFAST>
__device__ __noinline__ void gen_fft_pass_odd(const cd* a, cd* b, int L, FastDiv fL, FastDiv fL0, int S0, int S1, int SE, int n,
                                              GenPass ps, const cd* __restrict__ twN) {
    gen_fft_pass<R, S, LFAST>(a, b, L, fL, fL0, S0, S1, SE, n, ps, twN);
}

// The same transform over L lines whose starts follow a two-level pattern: line l begins at
// (l / L0) * S1 + (l % L0) * S0 (stacked planes of strided columns, or stacked rows), element stride SE.  Every
// division is a multiply-high with constants from the host.  Inlined into the caller, so that a, b and twN keep
// their shared-memory address space (LDS / STS, not generic accesses) and the plan is read straight from the
// kernel's parameter bank: through an out-of-line call with generic pointers a pass on a handful of lines took
// ~900 cycles, most of it address-space and parameter overhead.
// BIG: the plan may also hold passes of radix 8 and 16 (kernels_gen.cu; kernels_small.cu keeps to 2 and 4 for its
// instruction-cache footprint).
template <int S, bool LFAST, bool BIG = false>
__device__ __forceinline__ cd* gen_fft_lines2(cd* a, cd* b, int L, FastDiv fL, FastDiv fL0, int S0, int S1, int SE, const GenPlanP& pl,
                                              const cd* __restrict__ twN) {
    for (int s = 0; s < pl.nfac; ++s) {
        const GenPass ps = pl.pass[s];
        if (BIG && ps.r == 16) gen_fft_pass<16, S, LFAST>(a, b, L, fL, fL0, S0, S1, SE, pl.n, ps, twN);
        else if (BIG && ps.r == 8) gen_fft_pass<8, S, LFAST>(a, b, L, fL, fL0, S0, S1, SE, pl.n, ps, twN);
        else switch (ps.r) {
            case 2: gen_fft_pass<2, S, LFAST>(a, b, L, fL, fL0, S0, S1, SE, pl.n, ps, twN); break;
            case 4: gen_fft_pass<4, S, LFAST>(a, b, L, fL, fL0, S0, S1, SE, pl.n, ps, twN); break;
            case 3: gen_fft_pass_odd<3, S, LFAST>(a, b, L, fL, fL0, S0, S1, SE, pl.n, ps, twN); break;
            case 5: gen_fft_pass_odd<5, S, LFAST>(a, b, L, fL, fL0, S0, S1, SE, pl.n, ps, twN); break;
            default: gen_fft_pass_odd<7, S, LFAST>(a, b, L, fL, fL0, S0, S1, SE, pl.n, ps, twN); break;
        }
        __syncthreads();
        cd* t = a; a = b; b = t;
    }
    return a;
}
