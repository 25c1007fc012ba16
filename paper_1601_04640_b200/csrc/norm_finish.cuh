// norm_finish.cuh — calcnorm: from per-block partial sums of |psi|^2 to the deferred norm factor of
// every batch member, by the last block to finish.  Shared by kernels_cn.cu and kernels_gen.cu (product path only).
#pragma once
#include "dbec_internal.hpp"

// The last block to finish adds the per-block partial sums in index order and writes the deferred
// norm factor s = 1/sqrt(dV sum |psi|^2) of every batch member   (calcnorm; reading S13).  The blocks of a
// member are consecutive: member m owns partial[m*bpm .. (m+1)*bpm), bpm = blocks / nb.  One member: the
// whole block sums; a batch: one warp per member.  Fixed order either way (bit-reproducible).
__device__ __forceinline__ void norm_finish(double part, double* __restrict__ partial, unsigned int* ticket,
                                            double* __restrict__ scal, double dV, double* red, int nb) {
    __shared__ bool last;
    const unsigned int nblk = gridDim.x * gridDim.y;
    const unsigned int b = blockIdx.y * gridDim.x + blockIdx.x;
    if (threadIdx.x == 0) {
        partial[b] = part;
        __threadfence();
        last = (atomicAdd(ticket, 1u) == nblk - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    if (nb == 1) {
        double acc = 0.0;
        for (unsigned int i = threadIdx.x; i < nblk; i += blockDim.x) acc += __ldcg(partial + i);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        __syncthreads();
        if (l == 0) red[w] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int i = 0; i < nw; ++i) tot += red[i];
            const double s = 1.0 / sqrt(tot * dV);
            scal[SC_S] = s;
            scal[SC_S2] = s * s;
        }
    } else {
        const unsigned int bpm = nblk / nb;
        for (int m = w; m < nb; m += nw) {
            double acc = 0.0;
            for (unsigned int i = l; i < bpm; i += 32) acc += __ldcg(partial + (size_t)m * bpm + i);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
            if (l == 0) {
                const double s = 1.0 / sqrt(acc * dV);
                scal[(size_t)m * SC_COUNT + SC_S] = s;
                scal[(size_t)m * SC_COUNT + SC_S2] = s * s;
            }
        }
    }
    if (threadIdx.x == 0) *ticket = 0u;
}

