// tma_pipe.cuh — sm_100a asynchronous-copy plumbing for the persistent tile kernels: mbarriers, TMA
// tensor loads/stores (cp.async.bulk.tensor), 1-D bulk copies (cp.async.bulk), proxy fences and named
// barriers, as thin inline-PTX wrappers.  Product path only; nothing here is used by oracle/.
//
// Pattern (every persistent kernel in kernels_tma.cu / kernels_xline.cu):
//   loader thread   waits empty[s], arms full[s] with the tile's byte count, issues the TMA loads
//   worker groups   wait full[s], transform the tile in shared memory, fence.proxy.async, arrive done[s]
//   storer threads  (two: even / odd stages) wait done[s], issue the TMA store, and free the stage
//                   (arrive empty[s]) once the store has finished READING shared memory
//                   (cp.async.bulk.wait_group.read); a stage always belongs to the same storer
// so that global loads, arithmetic and global stores of different tiles overlap inside one CTA.
#pragma once
#include <cuda.h>
#include "dbec_internal.hpp"
#include <stdint.h>
#include <utility>

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity), "r"(0x989680u)     // suspend-time hint: sleep in hardware, do not spin
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ bool mbar_test_wait(uint64_t* bar, uint32_t parity) {      // never blocks
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {}
}

// ---- loader -> workers: number of tiles whose loads have been issued ----
// A worker may only wait on full[s] for the k-th use of stage s once the (k-1)-th use has landed:
// mbarrier waits test a phase PARITY, so a worker that runs a whole ring ahead of its stage would
// otherwise see the parity of an older, completed phase and walk into a stage that is still in use.
// The loader publishes its tile counter after it has passed empty[s]; workers check it first.
__device__ __forceinline__ int ld_acquire_shared(const int* p) {
    int v;
    asm volatile("ld.acquire.cta.shared::cta.b32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_shared(int* p, int v) {
    asm volatile("st.release.cta.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void wait_issued(const int* issued, int i) {
    while (ld_acquire_shared(issued) <= i) __nanosleep(64);
}

// generic-proxy writes to shared memory become visible to the async proxy (TMA store reads them)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- tensor-map copies (3-D maps; coordinates innermost first) ----
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, int c0, int c1, int c2, const void* src) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
                 ::"l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}

// ---- L2 eviction policies (createpolicy + .L2::cache_hint on every bulk / TMA access) ----
// What stays in the 126 MB L2 at the end of a pass should be its OUTPUT, which the next pass walks first
// (TileGeom::rev): outputs of the x-line kernels are stored evict-last, inputs that nobody reads again soon
// (the spectrum in the x-line kernel, psi in the density kernel, the V_dd tiles) are loaded evict-first,
// every other access carries a neutral hint.  Measured alternatives: profiles/r1d_step_ncu_full.md.
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// Policy from a code (dbec_handle_s::pol): c >= 2 evict-first; otherwise a fraction c (0..1) of the lines
// evict-last and the rest left alone (c = 0: neutral, c = 1: all evict-last).
__device__ __forceinline__ uint64_t l2_policy_code(float c) {
    if (c >= 2.f) return l2_policy_evict_first();
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.L2::evict_unchanged.b64 %0, %1;" : "=l"(pol) : "f"(c));
    return pol;
}
__device__ __forceinline__ void tma_store_3d_hint(const CUtensorMap* map, int c0, int c1, int c2, const void* src, uint64_t pol) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3, %4}], [%1], %5;"
                 ::"l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void bulk_store_hint(void* dst, const void* src, uint32_t bytes, uint64_t pol) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void tma_load_3d_hint(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar,
                                                 uint64_t pol) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)), "l"(pol)
        : "memory");
}
__device__ __forceinline__ void bulk_load_hint(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
                 : "memory");
}

// ---- 1-D bulk copies (contiguous runs, multiples of 16 bytes, 16-byte aligned on both sides) ----
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N> __device__ __forceinline__ void bulk_wait() {
    asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}

// ---- programmatic dependent launch: a kernel launched with launch_pdl() may become resident while the
// kernel before it in the stream is still draining; everything it does before pdl_wait() (staging constant
// tables, initialising barriers) overlaps that tail, everything after sees the predecessor's memory ----
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---- pacing of a loader thread against the wall clock ----
// A pass that streams a field much larger than L2 runs fastest when the CTAs walk their tiles in lockstep: the
// tiles neighbouring CTAs work on at the same moment are neighbours in memory (128-byte pieces of the same rows), and
// DRAM serves them from open pages.  Left alone, CTAs whose workers are quicker than their share of the memory
// bandwidth drift apart, every piece opens its page again, and the pass drops to 0.77 - 0.85 of the copy bandwidth
// (measured at 512 x 512 x 256: the imaginary-time y sweep, with LESS arithmetic per tile, took 423 us where the
// real-time one took 333).  So every loader issues its tile i on a schedule: head_ns apart for the first `head`
// tiles (what the previous pass left in L2, kernels_tma.cu: set_pace), pace_ns apart after that — the time the whole
// grid needs for one tile each at a bandwidth just below what DRAM sustains (dbec_handle_s::pace_gbs).  The
// schedule has to BIND at all times (a slack of two tiles lets the CTAs drift inside it and loses the effect) and it
// has to be COMMON: a CTA that finds itself late publishes by how much (atomicMax on one word in global memory),
// and every loader adds that lag to its own schedule, so the pack moves at the pace of its slowest member instead
// of falling apart when the schedule is too optimistic.  The last loader to finish clears the word for the next
// launch (launches that use it are ordered by the stream; their loaders start after griddepcontrol.wait).
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void pace_wait(unsigned long long& t0, int i, int head, int head_ns, int pace_ns, PaceState* ps) {
    if (i == 0) { t0 = global_ns(); return; }
    const unsigned long long nominal = t0 + (unsigned long long)(i < head ? i : head) * (unsigned long long)head_ns +
                                       (unsigned long long)(i > head ? i - head : 0) * (unsigned long long)pace_ns;
    const unsigned long long lag = ld_relaxed_u64(&ps->lag);
    const unsigned long long now = global_ns();
    if (now > nominal + lag + (unsigned long long)(pace_ns >> 3)) atomicMax(&ps->lag, now - nominal);     // late: everyone waits for me
    else while (global_ns() < nominal + lag) __nanosleep(40);
}
__device__ __forceinline__ void pace_wait(unsigned long long& t0, int i, const PaceArgs& pa) {
    pace_wait(t0, i, pa.head, pa.head_ns, pa.ns, pa.st);
}
__device__ __forceinline__ void pace_done(PaceState* ps) {
    __threadfence();
    if (atomicAdd(&ps->exits, 1u) == gridDim.x - 1) { ps->lag = 0ull; ps->exits = 0u; __threadfence(); }
}

// barrier over `nthreads` threads (a multiple of 32) with hardware barrier `id` (1..15; 0 is __syncthreads)
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

#if defined(__CUDACC__)
// Host: launch with programmatic stream serialisation (the kernel MUST call pdl_wait() before it touches
// anything an earlier kernel of the stream writes).
template <class K, class... Args>
static inline cudaError_t launch_pdl(K kernel, dim3 grid, dim3 block, size_t smem, cudaStream_t stream, int enable, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = enable ? 1 : 0;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
#endif
