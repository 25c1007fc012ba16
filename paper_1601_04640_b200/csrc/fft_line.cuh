// fft_line.cuh — register-resident line FFT of length N = 16*R2*R3 in complex128.
//
// The DFT of PAPER.md:63 ("Fourier transformation to momentum space") along one grid line.
// T = R2*R3 = N/16 threads own one line; thread m holds 16 values in registers.
//   on entry  v[j] = x[j*T + m]        on exit  v[j] = X[j*T + m]
// so a forward transform, a pointwise multiply and an inverse transform chain with no extra exchange.
//
// Cooley-Tukey index maps (n = input index, k = output index):
//   n = n1*T + n2*R3 + n3,  k = k1 + 16*k2 + 16*R2*k3
//   stage 1: 16-point DFT over n1 in registers, twiddle W_N^{(n2*R3+n3) k1}
//   stage 2: R2-point DFT over n2 (operands exchanged through shared memory), twiddle W_T^{n3 k2}
//   stage 3: R3-point DFT over n3 (second exchange), only when R3 > 1
// Every function is __host__ __device__ so the index maps can be exercised on the CPU.
#pragma once
#include "cplx.cuh"

// ---- small DFTs, natural order in and out, S = -1 forward / +1 inverse ----

template <int S> DBEC_HD void dft2(cd& a0, cd& a1) {
    cd t = a0;
    a0 = cadd(t, a1);
    a1 = csub(t, a1);
}

template <int S> DBEC_HD void dft4(cd& a0, cd& a1, cd& a2, cd& a3) {
    cd t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = cmul_si<S>(csub(a1, a3));
    a0 = cadd(t0, t2);
    a1 = cadd(t1, t3);
    a2 = csub(t0, t2);
    a3 = csub(t1, t3);
}

template <int S> DBEC_HD void dft8(cd& a0, cd& a1, cd& a2, cd& a3, cd& a4, cd& a5, cd& a6, cd& a7) {
    const double r = 0.70710678118654752440;
    dft4<S>(a0, a2, a4, a6);   // E[0..3] in a0,a2,a4,a6
    dft4<S>(a1, a3, a5, a7);   // O[0..3] in a1,a3,a5,a7
    cd o1 = cmake(r * (a3.x - S * a3.y), r * (S * a3.x + a3.y));      // O1 * W8^1
    cd o2 = cmul_si<S>(a5);                                           // O2 * W8^2
    cd o3 = cmake(r * (-a7.x - S * a7.y), r * (S * a7.x - a7.y));     // O3 * W8^3
    cd e0 = a0, e1 = a2, e2 = a4, e3 = a6, o0 = a1;
    a0 = cadd(e0, o0); a4 = csub(e0, o0);
    a1 = cadd(e1, o1); a5 = csub(e1, o1);
    a2 = cadd(e2, o2); a6 = csub(e2, o2);
    a3 = cadd(e3, o3); a7 = csub(e3, o3);
}

template <int S> DBEC_HD void dft16(cd (&v)[16]) {
    const double c1 = 0.92387953251128675613, s1 = 0.38268343236508977173;   // cos, sin(pi/8)
    const double r = 0.70710678118654752440;
    dft8<S>(v[0], v[2], v[4], v[6], v[8], v[10], v[12], v[14]);   // E[k] in v[2k]
    dft8<S>(v[1], v[3], v[5], v[7], v[9], v[11], v[13], v[15]);   // O[k] in v[2k+1]
    cd o[8];
    o[0] = v[1];
    o[1] = cmul(v[3], cmake(c1, S * s1));
    o[2] = cmake(r * (v[5].x - S * v[5].y), r * (S * v[5].x + v[5].y));
    o[3] = cmul(v[7], cmake(s1, S * c1));
    o[4] = cmul_si<S>(v[9]);
    o[5] = cmul(v[11], cmake(-s1, S * c1));
    o[6] = cmake(r * (-v[13].x - S * v[13].y), r * (S * v[13].x - v[13].y));
    o[7] = cmul(v[15], cmake(-c1, S * s1));
    cd e[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) e[k] = v[2 * k];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        v[k] = cadd(e[k], o[k]);
        v[k + 8] = csub(e[k], o[k]);
    }
}

template <int R, int S> DBEC_HD void dft_small(cd* w) {
    if (R == 2) dft2<S>(w[0], w[1]);
    else if (R == 4) dft4<S>(w[0], w[1], w[2], w[3]);
    else if (R == 8) dft8<S>(w[0], w[1], w[2], w[3], w[4], w[5], w[6], w[7]);
    else if (R == 16) {
        cd(&a)[16] = *reinterpret_cast<cd(*)[16]>(w);
        dft16<S>(a);
    }
}

// ---- plan ----

// PAD: pad the exchange rows so that a line stored contiguously (element stride 1) is read without
// bank conflicts; not needed when lines are interleaved column-wise (element stride = tile width).
template <int R2_, int R3_, bool PAD_ = true> struct FftPlan {
    static constexpr int R2 = R2_, R3 = R3_;
    static constexpr int T = R2_ * R3_;          // threads per line
    static constexpr int N = 16 * T;             // line length
    static constexpr int P1 = T + (PAD_ ? R3_ : 0);   // row pitch of the stage-1 exchange
    static constexpr int P3 = R3_ + (PAD_ ? 1 : 0);   // row pitch of the stage-2 exchange
    static constexpr int I2 = 16 / R2_;          // radix-R2 butterflies per thread in stage 2
    static constexpr int I3 = 16 / R3_;          // radix-R3 butterflies per thread in stage 3
    // shared-memory elements one line needs
    static constexpr int SMEM_A = 16 * P1, SMEM_B = (R3_ > 1) ? 16 * R2_ * P3 : 0;
    static constexpr int SMEM = (T == 1) ? 1 : (SMEM_A > SMEM_B ? SMEM_A : SMEM_B);
};

// stage 1: 16-point DFT over n1 and twiddle by W_N^{m k1}; twA[k1*T + m] = exp(-2 pi i m k1 / N).
template <class P, int S> DBEC_HD void fft_stage1(cd (&v)[16], int m, const cd* __restrict__ twA) {
    dft16<S>(v);
    if (P::T > 1) {
#pragma unroll
        for (int k1 = 1; k1 < 16; ++k1) v[k1] = cmul(v[k1], tw_dir<S>(twA[k1 * P::T + m]));
    }
}

// exchange 1, write: element (k1, m) at (k1*P1 + m)*es
template <class P> DBEC_HD void fft_x1_write(const cd (&v)[16], int m, cd* sm, int es) {
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) sm[(k1 * P::P1 + m) * es] = v[k1];
}

// stage 2: I2 butterflies of radix R2 per thread.  R3 == 1: final, v[j] = X[j*T + m].
// R3 > 1: v[i*R2 + k2] holds the twiddled value for item q = m + T*i (k1 = q / R3, n3 = q % R3).
// twN[j] = exp(-2 pi i j / N).
template <class P, int S> DBEC_HD void fft_stage2(cd (&v)[16], int m, const cd* sm, int es,
                                                  const cd* __restrict__ twN) {
    cd w[P::R2];
#pragma unroll
    for (int i = 0; i < P::I2; ++i) {
        const int q = m + P::T * i;
        const int n3 = q % P::R3, k1 = q / P::R3;
#pragma unroll
        for (int n2 = 0; n2 < P::R2; ++n2) w[n2] = sm[(k1 * P::P1 + n2 * P::R3 + n3) * es];
        dft_small<P::R2, S>(w);
        if (P::R3 == 1) {
#pragma unroll
            for (int k2 = 0; k2 < P::R2; ++k2) v[i + P::I2 * k2] = w[k2];
        } else {
            v[i * P::R2] = w[0];
#pragma unroll
            for (int k2 = 1; k2 < P::R2; ++k2)
                v[i * P::R2 + k2] = cmul(w[k2], tw_dir<S>(twN[16 * n3 * k2]));
        }
    }
}

// exchange 2, write (R3 > 1): element (p = k1 + 16*k2, n3) at (p*P3 + n3)*es
template <class P> DBEC_HD void fft_x2_write(const cd (&v)[16], int m, cd* sm, int es) {
#pragma unroll
    for (int i = 0; i < P::I2; ++i) {
        const int q = m + P::T * i;
        const int n3 = q % P::R3, k1 = q / P::R3;
#pragma unroll
        for (int k2 = 0; k2 < P::R2; ++k2) sm[((k1 + 16 * k2) * P::P3 + n3) * es] = v[i * P::R2 + k2];
    }
}

// stage 3 (R3 > 1): I3 butterflies of radix R3 per thread; final, v[j] = X[j*T + m].
template <class P, int S> DBEC_HD void fft_stage3(cd (&v)[16], int m, const cd* sm, int es) {
    cd w[P::R3 > 1 ? P::R3 : 2];
#pragma unroll
    for (int i = 0; i < P::I3; ++i) {
        const int p = m + P::T * i;
#pragma unroll
        for (int n3 = 0; n3 < P::R3; ++n3) w[n3] = sm[(p * P::P3 + n3) * es];
        dft_small<P::R3, S>(w);
#pragma unroll
        for (int k3 = 0; k3 < P::R3; ++k3) v[i + P::I3 * k3] = w[k3];
    }
}

#if defined(__CUDACC__)
// One line FFT in registers with its shared-memory exchanges.  SYNC = 0: the T threads of a line sit
// in one warp (__syncwarp); SYNC = 1: block-wide barrier (tile kernels).
template <class P, int S, int SYNC>
__device__ __forceinline__ void fft_line(cd (&v)[16], int m, cd* sm, int es, const cd* __restrict__ twA,
                                         const cd* __restrict__ twN) {
    fft_stage1<P, S>(v, m, twA);
    if (P::T > 1) {
        fft_x1_write<P>(v, m, sm, es);
        if (SYNC) __syncthreads(); else __syncwarp();
        fft_stage2<P, S>(v, m, sm, es, twN);
        if (P::R3 > 1) {
            if (SYNC) __syncthreads(); else __syncwarp();
            fft_x2_write<P>(v, m, sm, es);
            if (SYNC) __syncthreads(); else __syncwarp();
            fft_stage3<P, S>(v, m, sm, es);
        }
    }
}
#endif
