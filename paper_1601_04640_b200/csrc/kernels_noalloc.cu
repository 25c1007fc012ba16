// kernels_noalloc.cu — calcnorm (the norm integral dV sum |psi|^2) for callers that may not allocate:
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// A variant of k_norm (kernels_cn.cu).  That kernel keeps its block partial sums and its last-block ticket in the
// workspace the caller of dbec_create hands over; this one keeps them in a file-scope device array of fixed size,
// so the entry point needs no handle and no workspace and calls no cudaMalloc, cudaFree or allocating routine.
//
//   * The array costs DBEC_NOALLOC_SCRATCH_BYTES (about 256 KiB) on EVERY GPU that loads the library, until exit.
//   * One partial sum per block of NOALLOC_POINTS_PER_BLOCK points, so a call takes at most DBEC_NOALLOC_MAX_POINTS
//     points (2^27: twice BASELINE.json's largest grid, 512 x 512 x 256); more is refused with DBEC_ENOALLOC_SIZE.
//   * Every call on a device shares the array, which keeps the last call's contents.  The only word that must start
//     at zero, the ticket, is cleared on the caller's stream before each launch.  Calls that OVERLAP on the GPU
//     (different streams, or several host threads) race on the array: run them on one stream, or serialise them.
//   * In host code the array's name is a host-side stand-in, not a device address; the address comes from
//     cudaGetSymbolAddress, asked once per device with that device current.
// Fixed summation order (block partials of fixed extent, summed in index order by the last block): the result does
// not depend on the number of SMs or on the order in which blocks finish.
#include <cuda_runtime.h>
#include <mutex>
#include "dbec_internal.hpp"
#include "cplx.cuh"

constexpr int NOALLOC_THREADS = 256;
constexpr int NOALLOC_POINTS_PER_BLOCK = 4096;                      // 16 points per thread
constexpr int NOALLOC_MAX_PARTIALS = (int)(DBEC_NOALLOC_MAX_POINTS / NOALLOC_POINTS_PER_BLOCK);   // 32768
constexpr int NOALLOC_TICKET_WORDS = 64;                            // the ticket has 256 bytes to itself
static_assert(DBEC_NOALLOC_MAX_POINTS % NOALLOC_POINTS_PER_BLOCK == 0, "whole blocks");
static_assert(DBEC_NOALLOC_SCRATCH_BYTES == NOALLOC_MAX_PARTIALS * sizeof(double) + NOALLOC_TICKET_WORDS * sizeof(unsigned int),
              "the size include/dbec.h states");

struct NoallocScratch {
    double partial[NOALLOC_MAX_PARTIALS];
    unsigned int ticket[NOALLOC_TICKET_WORDS];
};
static __device__ __align__(256) NoallocScratch noalloc_scratch;

// Sum over the block in a fixed order (warp shuffles, then warp 0 over the warp sums); valid in thread 0.
__device__ __forceinline__ double noalloc_block_sum(double x, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) red[w] = x;
    __syncthreads();
    double t = (threadIdx.x < NOALLOC_THREADS / 32) ? red[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;
}

// Block b sums points [b * 4096, (b + 1) * 4096); the last block to finish adds the partials up and writes
// dV * sum to *out.  s: the scratch (the address of noalloc_scratch on this device).
__global__ void __launch_bounds__(NOALLOC_THREADS)
k_norm_noalloc(const cd* __restrict__ psi, long long P, double dV, NoallocScratch* s, double* __restrict__ out) {
    __shared__ double red[32];
    __shared__ bool last;
    const long long base = (long long)blockIdx.x * NOALLOC_POINTS_PER_BLOCK;
    double acc = 0.0;
#pragma unroll 4
    for (int k = 0; k < NOALLOC_POINTS_PER_BLOCK / NOALLOC_THREADS; ++k) {
        const long long i = base + k * NOALLOC_THREADS + threadIdx.x;
        if (i < P) acc += cnorm2(psi[i]);
    }
    const double part = noalloc_block_sum(acc, red);
    if (threadIdx.x == 0) {
        s->partial[blockIdx.x] = part;
        __threadfence();
        last = (atomicAdd(s->ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double a = 0.0;
    for (unsigned int i = threadIdx.x; i < gridDim.x; i += NOALLOC_THREADS) a += __ldcg(s->partial + i);
    const double tot = noalloc_block_sum(a, red);
    if (threadIdx.x == 0) {
        *out = tot * dV;
        s->ticket[0] = 0u;
    }
}

// The device address of the scratch array, asked once per device with that device current.
static int noalloc_scratch_ptr(NoallocScratch** out) {
    constexpr int MAXDEV = 64;
    static std::mutex mu;
    static NoallocScratch* ptr[MAXDEV] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    if (dev < 0 || dev >= MAXDEV) return (int)cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        NoallocScratch* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, noalloc_scratch);
        if (e != cudaSuccess) return (int)e;
        if (!p) return (int)cudaErrorInvalidSymbol;
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return 0;
}

static thread_local int noalloc_cuda_error = 0;

extern "C" int dbec_norm_noalloc(const void* psi_c128_dev, long long npoints, double dV, double* norm_dev, void* cuda_stream) {
    noalloc_cuda_error = 0;
    if (!psi_c128_dev || !norm_dev || npoints < 1 || !(dV > 0.0)) return DBEC_EINVAL;
    if (npoints > DBEC_NOALLOC_MAX_POINTS) return DBEC_ENOALLOC_SIZE;
    NoallocScratch* s = nullptr;
    int rc = noalloc_scratch_ptr(&s);
    if (rc) { noalloc_cuda_error = rc; return DBEC_ECUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the ticket must start at zero whatever an earlier (possibly failed) call left behind
    cudaError_t e = cudaMemsetAsync(s->ticket, 0, sizeof(s->ticket), st);
    if (e != cudaSuccess) { noalloc_cuda_error = (int)e; return DBEC_ECUDA; }
    const int nblk = (int)((npoints + NOALLOC_POINTS_PER_BLOCK - 1) / NOALLOC_POINTS_PER_BLOCK);
    k_norm_noalloc<<<nblk, NOALLOC_THREADS, 0, st>>>((const cd*)psi_c128_dev, npoints, dV, s, norm_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) { noalloc_cuda_error = (int)e; return DBEC_ECUDA; }
    return DBEC_OK;
}

extern "C" int dbec_noalloc_last_cuda_error(void) { return noalloc_cuda_error; }
