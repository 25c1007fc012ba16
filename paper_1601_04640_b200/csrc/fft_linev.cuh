// fft_linev.cuh — register-resident line FFT of length N = V*R2*R3 with V = 8 or 16 values per thread.
//
// Same transform and the same index maps as fft_line.cuh (the DFT of PAPER.md:63 along one grid line), with the
// number of values a thread holds as a parameter, so that a line of 256 points can be owned by the 32 lanes of
// ONE warp (V = 8, T = 32): every exchange is then a __syncwarp, no block-level barrier.
//   T = R2*R3 = N/V threads per line;  on entry v[j] = x[j*T + m],  on exit v[j] = X[j*T + m]   (j < V)
//   n = n1*T + n2*R3 + n3,  k = k1 + V*k2 + V*R2*k3
//   stage 1: V-point DFT over n1 in registers, twiddle W_N^{m k1}, m = n2*R3 + n3
//   stage 2: R2-point DFT over n2 (operands exchanged through shared memory), twiddle W_T^{n3 k2}
//   stage 3: R3-point DFT over n3 (second exchange), only when R3 > 1
// Every function is __host__ __device__ so the index maps can be exercised on the CPU.
#pragma once
#include "fft_line.cuh"

template <int V_, int R2_, int R3_> struct FftPlanV {
    static constexpr int V = V_, R2 = R2_, R3 = R3_;
    static constexpr int T = R2_ * R3_;              // threads per line
    static constexpr int N = V_ * T;                 // line length
    static constexpr int P1 = T + R3_;               // row pitch of the stage-1 exchange (conflict-free stage-2 reads)
    static constexpr int P3 = R3_;                   // row pitch of the stage-2 exchange; entry (p, n3) sits at
                                                     // p*R3 + (n3 ^ x2_rot(p)): conflict-free both ways (x2_pos)
    static constexpr int I2 = V_ / R2_;              // radix-R2 butterflies per thread in stage 2
    static constexpr int I3 = V_ / R3_;              // radix-R3 butterflies per thread in stage 3
    static constexpr int SMEM_A = V_ * P1, SMEM_B = (R3_ > 1) ? V_ * R2_ * P3 : 0;
    static constexpr int SMEM = SMEM_A > SMEM_B ? SMEM_A : SMEM_B;   // shared-memory elements one line needs
    static_assert(V_ % R2_ == 0 && V_ % R3_ == 0, "stage radices must divide the values per thread");
};

// Stage-2 exchange position of entry (p, n3).  R3 = 4: rows of 4 x 16 bytes; rotating the entry index by
// bits 1..2 of the row puts the 8 rows a quarter warp touches (writes: 2 rows x 4 entries; reads: 8 rows, same
// entry) into 8 different 16-byte bank groups.  R3 = 2: rows of 2, rotation by bit 2 of the row.  R3 = 8: rows of
// 8 x 16 bytes = all bank groups; rotating by the row index keeps a row's writes a permutation of the row and sends
// the 8 rows a quarter warp reads (same entry) to 8 different groups (plain: an 8-way conflict).
template <class P> DBEC_HD int x2_pos(int p, int n3) {
    return P::R3 == 8 ? p * 8 + ((n3 + p) & 7)
         : P::R3 == 4 ? p * 4 + (n3 ^ ((p >> 1) & 3)) : P::R3 == 2 ? p * 2 + (n3 ^ ((p >> 2) & 1)) : p * P::R3 + n3;
}

template <int V, int S> DBEC_HD void dft_regs(cd (&v)[V]) { dft_small<V, S>(v); }

// twA[k1*T + m] = exp(-2 pi i m k1 / N)
template <class P, int S> DBEC_HD void fftv_stage1(cd (&v)[P::V], int m, const cd* __restrict__ twA) {
    dft_regs<P::V, S>(v);
#pragma unroll
    for (int k1 = 1; k1 < P::V; ++k1) v[k1] = cmul(v[k1], tw_dir<S>(twA[k1 * P::T + m]));
}

template <class P> DBEC_HD void fftv_x1_write(const cd (&v)[P::V], int m, cd* sm) {
#pragma unroll
    for (int k1 = 0; k1 < P::V; ++k1) sm[k1 * P::P1 + m] = v[k1];
}

// tw2[k2*R3 + n3] = exp(-2 pi i V n3 k2 / N): the R2*R3 stage-2 twiddles; the R3 entries the lanes of a warp read
// in one instruction are neighbours (one wavefront)
template <class P, int S> DBEC_HD void fftv_stage2(cd (&v)[P::V], int m, const cd* sm, const cd* __restrict__ tw2) {
    cd w[P::R2];
#pragma unroll
    for (int i = 0; i < P::I2; ++i) {
        const int q = m + P::T * i;
        const int n3 = q % P::R3, k1 = q / P::R3;
#pragma unroll
        for (int n2 = 0; n2 < P::R2; ++n2) w[n2] = sm[k1 * P::P1 + n2 * P::R3 + n3];
        dft_small<P::R2, S>(w);
        if (P::R3 == 1) {
#pragma unroll
            for (int k2 = 0; k2 < P::R2; ++k2) v[i + P::I2 * k2] = w[k2];
        } else {
            v[i * P::R2] = w[0];
#pragma unroll
            for (int k2 = 1; k2 < P::R2; ++k2) v[i * P::R2 + k2] = cmul(w[k2], tw_dir<S>(tw2[k2 * P::R3 + n3]));
        }
    }
}

template <class P> DBEC_HD void fftv_x2_write(const cd (&v)[P::V], int m, cd* sm) {
#pragma unroll
    for (int i = 0; i < P::I2; ++i) {
        const int q = m + P::T * i;
        const int n3 = q % P::R3, k1 = q / P::R3;
#pragma unroll
        for (int k2 = 0; k2 < P::R2; ++k2) sm[x2_pos<P>(k1 + P::V * k2, n3)] = v[i * P::R2 + k2];
    }
}

template <class P, int S> DBEC_HD void fftv_stage3(cd (&v)[P::V], int m, const cd* sm) {
    cd w[P::R3 > 1 ? P::R3 : 2];
#pragma unroll
    for (int i = 0; i < P::I3; ++i) {
        const int p = m + P::T * i;
#pragma unroll
        for (int n3 = 0; n3 < P::R3; ++n3) w[n3] = sm[x2_pos<P>(p, n3)];
        dft_small<P::R3, S>(w);
#pragma unroll
        for (int k3 = 0; k3 < P::R3; ++k3) v[i + P::I3 * k3] = w[k3];
    }
}

#if defined(__CUDACC__)
// The T threads of a line sit in one warp: every exchange is a __syncwarp.
template <class P, int S>
__device__ __forceinline__ void fftv_line_warp(cd (&v)[P::V], int m, cd* sm, const cd* __restrict__ twA, const cd* __restrict__ tw2) {
    fftv_stage1<P, S>(v, m, twA);
    fftv_x1_write<P>(v, m, sm);
    __syncwarp();
    fftv_stage2<P, S>(v, m, sm, tw2);
    if (P::R3 > 1) {
        __syncwarp();
        fftv_x2_write<P>(v, m, sm);
        __syncwarp();
        fftv_stage3<P, S>(v, m, sm);
    }
}
#endif
