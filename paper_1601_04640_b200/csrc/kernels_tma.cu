// kernels_tma.cu — the strided line passes (FFT along y/z on the half spectrum, Crank-Nicolson sweeps
// along y/z on psi) as persistent, warp-specialised sm_100a kernels fed by the tensor memory
// accelerator.  Same arithmetic as k_fft_strided / k_cn_strided (calcpsidd2, calcluy, calcluz —
// PAPER.md:63, :67, :71, :79); what changes is how a tile travels:
//
//   global --TMA load--> shared stage --worker group: registers, in-place in the stage--> TMA store
//
// A tile is 8 neighbouring lines (8 x 16 B = one 128-byte row per line point), N rows.  One CTA per SM
// walks its tiles round-robin; a loader thread keeps several stages in flight, NG worker groups each
// transform one tile at a time, a storer thread drains finished stages.  Loads, arithmetic and stores
// of different tiles overlap, so HBM stays busy while the Thomas recurrences and butterflies run.
#include "dbec_internal.hpp"
#include "fft_line.cuh"
#include "cn_chunk.cuh"
#include "cn_line_smem.cuh"
#include "tma_pipe.cuh"

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return (int)e_; } while (0)

constexpr int TCOLS = DBEC_SPEC_COLS;   // lines per tile

struct TileGeom {
    int ntiles_x;    // tiles along x (the contiguous direction)
    int ntiles;      // all tiles of the pass (of the slab)
    int axis;        // 1: lines along y, outer coordinate z;  2: lines along z, outer coordinate y
    int box_rows;    // rows of one TMA box (<= 256)
    int nbox;        // boxes per tile (N / box_rows)
    int outer0;      // first outer coordinate (slab offset; axis 1 only)
    int vfold;       // fused z pass: NY (the tile's outer coordinate k_y folds to min(k_y, NY - k_y) in the V_dd table);
                     // fused y pass of a 2-D grid: 0 (the table has one plane, shared by the members of a batch)
    int vrows;       // rows of one V_dd box, boxes per tile
    int vnbox;
    int pace_ns;     // interval at which the loader issues its tiles (tma_pipe.cuh: pace_wait; 0: no pacing)
    int pace_head, pace_head_ns;   // the first pace_head tiles of a CTA, which come out of L2, at this shorter interval
    PaceState* pace;               // the launch's shared lag word
    int ystep;       // z passes: rows of y per tile (1, or 2 when a tile is 8 columns x 2 rows of y: k_cn_tma with TC = 16)
    int rev;         // walk the tiles last to first (so that a pass starts on what the previous one left in L2)
    int fold_pairs;  // fused z pass: outer coordinates in the order 0, 1, NY-1, 2, NY-2, ... so that the two rows k_y and
                     // NY - k_y, which read the same V_dd tile, are worked on at the same time (the second read hits L2)
    float pol_ld, pol_st;   // L2 eviction policy codes of the tile loads / stores (tma_pipe.cuh: l2_policy_code)
};

struct PipeBars {
    uint64_t* full; uint64_t* empty; uint64_t* done;
    int* issued;     // tiles whose loads the loader has issued (tma_pipe.cuh: wait_issued)
};

template <int NST> __device__ __forceinline__ PipeBars pipe_init(uint64_t* bars, int done_count) {
    PipeBars b; b.full = bars; b.empty = bars + NST; b.done = bars + 2 * NST; b.issued = (int*)(bars + 3 * NST);
    if (threadIdx.x == 0) {
        *b.issued = 0;
        for (int s = 0; s < NST; ++s) { mbar_init(b.full + s, 1); mbar_init(b.empty + s, 1); mbar_init(b.done + s, done_count); }
        fence_mbar_init();
    }
    __syncthreads();
    pdl_launch_dependents();        // the next kernel of the stream may start its own prologue
    pdl_wait();                     // tables are staged, barriers set up: now wait for the previous kernel's data
    return b;
}

__device__ __forceinline__ void tile_coords(const TileGeom& tg, int t, int b, int inner, int& c0, int& c1, int& c2) {
    if (tg.rev) t = tg.ntiles - 1 - t;
    const int tx = t % tg.ntiles_x;
    int o = t / tg.ntiles_x + tg.outer0;
    if (tg.fold_pairs && o > 0) o = (o & 1) ? (o + 1) >> 1 : tg.fold_pairs - (o >> 1);
    c0 = tx * inner;
    c1 = tg.axis == 1 ? b * tg.box_rows : o * tg.ystep;
    c2 = tg.axis == 1 ? o : b * tg.box_rows;
}

// Loader: stage i % NST receives tile blockIdx.x + i * gridDim.x.  `extra` (optional) is a second
// tensor map whose box lands EXTRA_OFF bytes into the stage (the V_dd tile of the fused z pass).
// EXTRA_TX: the bytes the V_dd boxes really carry (EXTRA_BYTES includes the padding between them)
template <int NST, int STAGE_BYTES, int MAIN_BYTES, int EXTRA_BYTES, int EXTRA_TX = EXTRA_BYTES>
__device__ __forceinline__ void pipe_loader(const PipeBars& pb, unsigned char* stages, const CUtensorMap* map,
                                            const CUtensorMap* extra, const TileGeom& tg, int nmine) {
    const uint64_t pol = l2_policy_code(tg.pol_ld);
    unsigned long long t0 = 0;
    for (int i = 0; i < nmine; ++i) {
        const int s = i % NST;
        if (i >= NST) mbar_wait(pb.empty + s, ((i / NST) - 1) & 1);
        if (tg.pace_ns) pace_wait(t0, i, tg.pace_head, tg.pace_head_ns, tg.pace_ns, tg.pace);
        st_release_shared(pb.issued, i + 1);
        mbar_expect_tx(pb.full + s, MAIN_BYTES + EXTRA_TX);
        const int t = blockIdx.x + i * gridDim.x;
        unsigned char* dst = stages + (size_t)s * STAGE_BYTES;
        for (int b = 0; b < tg.nbox; ++b) {
            int c0, c1, c2;
            tile_coords(tg, t, b, 2 * TCOLS, c0, c1, c2);
            tma_load_3d_hint(dst + (size_t)b * (MAIN_BYTES / tg.nbox), map, c0, c1, c2, pb.full + s, pol);
        }
        if (EXTRA_BYTES) {
            // rows 0 .. N/2 of the folded V_dd table under this tile (table [nzf][nyf][nxhp]; 2-D: [1][nyf][nxhp]).
            // Evict-first: measured at C4, keeping the 17 MiB table in L2 (evict-last) makes this pass no faster
            // and costs the next one 3 us of the spectrum lines it would otherwise find there.
            int c0, c1, c2;
            tile_coords(tg, t, 0, TCOLS, c0, c1, c2);
            const int o = tg.axis == 1 ? c2 : c1;
            const uint64_t polv = l2_policy_evict_first();
            for (int b = 0; b < tg.vnbox; ++b) {
                if (tg.vfold) tma_load_3d_hint(dst + MAIN_BYTES + (size_t)b * (EXTRA_BYTES / tg.vnbox), extra, c0,
                                               o < tg.vfold - o ? o : tg.vfold - o, b * tg.vrows, pb.full + s, polv);
                else tma_load_3d_hint(dst + MAIN_BYTES + (size_t)b * (EXTRA_BYTES / tg.vnbox), extra, c0, b * tg.vrows, 0,
                                      pb.full + s, polv);
            }
        }
    }    if (tg.pace_ns) pace_done(tg.pace);
}

// Two storers, one for the even and one for the odd stages (which = 0 / 1): while one sits in
// wait_group.read (which lasts about as long as the global write), the other already drains the next
// finished stage.  A stage always belongs to the same storer, so its done[] phases are seen in order.
template <int NST, int STAGE_BYTES, int MAIN_BYTES>
__device__ __forceinline__ void pipe_storer(const PipeBars& pb, unsigned char* stages, const CUtensorMap* map,
                                            const TileGeom& tg, int nmine, int which) {
    const uint64_t pol = l2_policy_code(tg.pol_st);
    for (int i = 0; i < nmine; ++i) {
        const int s = i % NST;
        if ((s & 1) != which) continue;
        mbar_wait(pb.done + s, (i / NST) & 1);
        const int t = blockIdx.x + i * gridDim.x;
        unsigned char* src = stages + (size_t)s * STAGE_BYTES;
        for (int b = 0; b < tg.nbox; ++b) {
            int c0, c1, c2;
            tile_coords(tg, t, b, 2 * TCOLS, c0, c1, c2);
            tma_store_3d_hint(map, c0, c1, c2, src + (size_t)b * (MAIN_BYTES / tg.nbox), pol);
        }
        bulk_commit();
        bulk_wait_read<0>();              // the copy engine has read the stage (takes about as long as the global write)
        mbar_arrive(pb.empty + s);
    }
    bulk_wait<0>();
}

// Sum over the block in a fixed order (same as kernels_cn.cu).
template <int NT> __device__ __forceinline__ double block_sum_t(double x, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    constexpr int NW = (NT + 31) / 32;
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) red[w] = x;
    __syncthreads();
    double t = (threadIdx.x < NW) ? red[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;   // valid in thread 0
}

// ------------------------------------------------------------------------------------------------
// Crank-Nicolson sweep along y or z (calcluy / calcluz)
// ------------------------------------------------------------------------------------------------
// TC: lines per tile — 8 neighbouring columns, or 16 = 8 columns x 2 neighbouring rows of y (z sweeps whose planes are
// 2 MiB or more apart: the two rows of a plane share a memory page, so a tile touches half as many pages per byte;
// measured at 512 x 512 x 256, plane stride 4 MiB: 473 -> 415 us; no change at 256^3, plane stride 1 MiB).
template <bool RT, int NCH, int NG, int NST, bool NORM, int TC>
__global__ void __launch_bounds__(NG* NCH* TC + 96, 1)
k_cn_tma(const __grid_constant__ CUtensorMap map, CnTab<RT> cn, TileGeom tg, double* __restrict__ partial,
         unsigned int* ticket, double* __restrict__ scal, double dV) {
    typedef typename CnCoef<RT>::type CT;
    constexpr int N = NCH * CN_L, GT = NCH * TC, TILE = N * TC, STAGE_BYTES = TILE * (int)sizeof(cd);
    constexpr int NT = NG * GT + 96;
    extern __shared__ __align__(1024) unsigned char smraw[];
    __shared__ double red[32];
    __shared__ bool last;
    unsigned char* base = smraw;     // (no integer round trip: the compiler must see shared-memory pointers)
    cd* ends = (cd*)(base + (size_t)NST * STAGE_BYTES);
    uint64_t* bars = (uint64_t*)(ends + NG * 2 * GT);
    // h / PF / PB (entry k at k + k/16, so that the four chunks a warp works on hit different banks) and
    // the chunk-end products, staged once per CTA: read straight from global memory inside the
    // recurrences every table value costs an exposed L1/L2 round trip
    CT* tab = (CT*)(bars + ((3 * NST + 3) & ~1));
    constexpr int E = cn_tab_elems(N);
    const int tid = threadIdx.x;
    CnTab<RT> cs = cn_stage_tables<RT, N>(cn, tab);
    for (int k = tid; k < NCH; k += NT) { tab[3 * E + k] = cn.pfe[k]; tab[3 * E + NCH + k] = cn.pbs[k]; }
    cs.pfe = tab + 3 * E; cs.pbs = tab + 3 * E + NCH;
    const PipeBars pb = pipe_init<NST>(bars, GT / 32);
    const int nmine = (tg.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    double acc = 0.0;
    if (tid < NG * GT) {
        const int g = tid / GT, r = tid % GT, col = r % TC, c = r / TC, j0 = c * CN_L;
        const int t0 = j0 + c;      // chunk c of the padded tables
        cd* myends = ends + g * 2 * GT;
        for (int i = g; i < nmine; i += NG) {
            const int s = i % NST;
            wait_issued(pb.issued, i);
            mbar_wait(pb.full + s, (i / NST) & 1);
            cd* t = (cd*)(base + (size_t)s * STAGE_BYTES) + col;
            cd u[CN_L];
#pragma unroll
            for (int k = 0; k < CN_L; ++k) u[k] = t[(j0 + k) * TC];
            const cd lo = (c > 0) ? t[(j0 - 1) * TC] : cmake(0.0, 0.0);
            const cd hi = (c < NCH - 1) ? t[(j0 + CN_L) * TC] : cmake(0.0, 0.0);
            cn_chunk_forward<CT>(u, lo, hi, cs.kap, cs.h + t0);
            myends[c * TC + col] = u[CN_L - 1];
            named_bar_sync(1 + g, GT);
            const cd din = cn_carry_forward<CT>(c, myends + col, TC, cs.pfe, cs.K);
            cn_chunk_backward<CT>(u, din, cs.h + t0, cs.pf + t0);
            myends[GT + c * TC + col] = u[0];
            named_bar_sync(1 + g, GT);
            const cd uin = cn_carry_backward<CT>(c, NCH, myends + GT + col, TC, cs.pbs, cs.K);
            cn_chunk_fix<CT>(u, uin, cs.pb + t0);
#pragma unroll
            for (int k = 0; k < CN_L; ++k) {
                t[(j0 + k) * TC] = u[k];
                if (NORM) acc += cnorm2(u[k]);
            }
            fence_proxy_async();
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(pb.done + s);
        }
    } else if (tid == NG * GT) {
        pipe_loader<NST, STAGE_BYTES, STAGE_BYTES, 0>(pb, base, &map, nullptr, tg, nmine);
    } else if (tid == NG * GT + 32 || tid == NG * GT + 64) {
        pipe_storer<NST, STAGE_BYTES, STAGE_BYTES>(pb, base, &map, tg, nmine, (tid - NG * GT) / 32 - 1);
    }
    if (NORM) {
        // calcnorm: block partial -> last block writes the deferred factor (reading S13)
        const double part = block_sum_t<NT>(acc, red);
        const unsigned int nb = gridDim.x;
        if (tid == 0) {
            partial[blockIdx.x] = part;
            __threadfence();
            last = (atomicAdd(ticket, 1u) == nb - 1);
        }
        __syncthreads();
        if (last) {
            __threadfence();
            double a = 0.0;
            for (unsigned int i = tid; i < nb; i += NT) a += __ldcg(partial + i);
            const double tot = block_sum_t<NT>(a, red);
            if (tid == 0) {
                const double sfac = 1.0 / sqrt(tot * dV);
                scal[SC_S] = sfac;
                scal[SC_S2] = sfac * sfac;
                *ticket = 0u;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// FFT along y or z on the half spectrum (calcpsidd2); MODE 2 = forward * V_dd(k)/P * inverse
// ------------------------------------------------------------------------------------------------
template <class P, int S>
__device__ __forceinline__ void fft_line_nb(cd (&v)[16], int m, cd* sm, const cd* __restrict__ twA,
                                            const cd* __restrict__ twN, int bar, int nthreads) {
    fft_stage1<P, S>(v, m, twA);
    if (P::T > 1) {
        fft_x1_write<P>(v, m, sm, TCOLS);            // every thread overwrites only rows it owns
        named_bar_sync(bar, nthreads);
        fft_stage2<P, S>(v, m, sm, TCOLS, twN);
        if (P::R3 > 1) {
            named_bar_sync(bar, nthreads);
            fft_x2_write<P>(v, m, sm, TCOLS);
            named_bar_sync(bar, nthreads);
            fft_stage3<P, S>(v, m, sm, TCOLS);
        }
    }
}

// Bytes of the V_dd part of a stage of the fused pass: rows 0 .. N/2 (N/2 + 1 rows of 8 doubles) in one box, or in
// two boxes of N/4 + 1 rows when that exceeds the 256 rows a box may have; rounded up to the 128 bytes a TMA
// destination must be aligned to.
__host__ __device__ constexpr int fmi_vrows(int n) { return n / 2 + 1 <= 256 ? n / 2 + 1 : n / 4 + 1; }
__host__ __device__ constexpr int fmi_vnbox(int n) { return n / 2 + 1 <= 256 ? 1 : 2; }
__host__ __device__ constexpr int fmi_extra_bytes(int n) {
    return fmi_vnbox(n) * ((fmi_vrows(n) * TCOLS * (int)sizeof(double) + 127) / 128 * 128);
}

template <class P, int MODE, int NG, int NST>
__global__ void __launch_bounds__(NG* P::T* TCOLS + 96, 1)
k_fft_tma(const __grid_constant__ CUtensorMap map, const __grid_constant__ CUtensorMap map_vdd,
          const cd* twA, const cd* twN, TileGeom tg) {
    constexpr int T = P::T, N = P::N, GT = T * TCOLS;
    constexpr int MAIN_BYTES = N * TCOLS * (int)sizeof(cd);
    constexpr int EXTRA_BYTES = (MODE == 2) ? fmi_extra_bytes(N) : 0;     // rows 0 .. N/2 of the folded V_dd table
    constexpr int STAGE_BYTES = MAIN_BYTES + EXTRA_BYTES;
    extern __shared__ __align__(1024) unsigned char smraw[];
    unsigned char* base = smraw;     // (no integer round trip: the compiler must see shared-memory pointers)
    uint64_t* bars = (uint64_t*)(base + (size_t)NST * STAGE_BYTES);
    // twiddle tables staged once per CTA (2 x N entries)
    cd* tw = (cd*)(bars + ((3 * NST + 3) & ~1));
    const int tid = threadIdx.x;
    for (int k = tid; k < N; k += NG * GT + 96) { tw[k] = twA[k]; tw[N + k] = twN[k]; }
    twA = tw; twN = tw + N;
    const PipeBars pb = pipe_init<NST>(bars, GT / 32);
    const int nmine = (tg.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    if (tid < NG * GT) {
        const int g = tid / GT, r = tid % GT, col = r % TCOLS, m = r / TCOLS;
        for (int i = g; i < nmine; i += NG) {
            const int s = i % NST;
            wait_issued(pb.issued, i);
            mbar_wait(pb.full + s, (i / NST) & 1);
            cd* sm = (cd*)(base + (size_t)s * STAGE_BYTES) + col;
            cd v[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = sm[(j * T + m) * TCOLS];
            if (MODE == 0 || MODE == 2) fft_line_nb<P, -1>(v, m, sm, twA, twN, 1 + g, GT);
            if (MODE == 2) {
                const double* w = (const double*)(base + (size_t)s * STAGE_BYTES + MAIN_BYTES) + col;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const int r = j * T + m, rf = r < N - r ? r : N - r;            // V_dd is even along the line
                    // (two boxes: the second one starts after the first one's padding)
                    constexpr int VR = fmi_vrows(N), PADR = fmi_extra_bytes(N) / fmi_vnbox(N) / (TCOLS * (int)sizeof(double)) - VR;
                    v[j] = cmul(w[(rf + (fmi_vnbox(N) > 1 && rf >= VR ? PADR : 0)) * TCOLS], v[j]);
                }
            }
            if (MODE == 2 && T > 1) named_bar_sync(1 + g, GT);      // stage-2/3 reads of the forward pass are over
            if (MODE == 1 || MODE == 2) fft_line_nb<P, +1>(v, m, sm, twA, twN, 1 + g, GT);
            if (T > 1) named_bar_sync(1 + g, GT);
#pragma unroll
            for (int j = 0; j < 16; ++j) sm[(j * T + m) * TCOLS] = v[j];
            fence_proxy_async();
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(pb.done + s);
        }
    } else if (tid == NG * GT) {
        pipe_loader<NST, STAGE_BYTES, MAIN_BYTES, EXTRA_BYTES, (MODE == 2 ? fmi_vnbox(N) * fmi_vrows(N) * TCOLS * (int)sizeof(double) : 0)>(
            pb, base, &map, &map_vdd, tg, nmine);
    } else if (tid == NG * GT + 32 || tid == NG * GT + 64) {
        pipe_storer<NST, STAGE_BYTES, MAIN_BYTES>(pb, base, &map, tg, nmine, (tid - NG * GT) / 32 - 1);
    }
}

// ------------------------------------------------------------------------------------------------
// tensor maps
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// A field of doubles [n2][n1][n0] (n0 fastest) and a box of (b0, b1, b2) elements.
static int make_map(CUtensorMap* m, void* ptr, long long n0, long long n1, long long n2, int b0, int b1, int b2,
                    bool swizzle128 = false) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return (int)cudaErrorNotSupported;
    cuuint64_t dims[3] = {(cuuint64_t)n0, (cuuint64_t)n1, (cuuint64_t)n2};
    cuuint64_t strides[2] = {(cuuint64_t)n0 * 8, (cuuint64_t)n0 * n1 * 8};
    cuuint32_t box[3] = {(cuuint32_t)b0, (cuuint32_t)b1, (cuuint32_t)b2};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, ptr, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : (int)cudaErrorInvalidValue;
}

static int box_rows_of(int n) { return n < 256 ? n : 256; }

// Maps of the handle: psi / spec / vdd, boxes along y and along z.  Called once by dbec_create.
int dbec_make_tensor_maps(dbec_handle_s* h) {
    static_assert(sizeof(CUtensorMap) == DBEC_TMAP_BYTES, "tensor map size");
    const int by = box_rows_of(h->ny), bz = box_rows_of(h->nz);
    int rc = 0;
    // psi and the spectrum hold nplanes = nz * nb planes (a batch of 2-D grids is a stack of planes; the
    // persistent strided kernels do not serve batches of 3-D grids, see dbec_tma_supported)
    const int np = h->nplanes;
    rc |= make_map((CUtensorMap*)h->tmap[TM_PSI_Y], h->psi, 2LL * h->nx, h->ny, np, 2 * TCOLS, by, 1);
    rc |= make_map((CUtensorMap*)h->tmap[TM_PSI_Z], h->psi, 2LL * h->nx, h->ny, np, 2 * TCOLS, 1, bz);
    if (h->ny % 2 == 0) rc |= make_map((CUtensorMap*)h->tmap[TM_PSI_Z2], h->psi, 2LL * h->nx, h->ny, np, 2 * TCOLS, 2, bz);
    rc |= make_map((CUtensorMap*)h->tmap[TM_SPEC_Y], h->spec, 2LL * h->nxhp, h->ny, np, 2 * TCOLS, by, 1);
    rc |= make_map((CUtensorMap*)h->tmap[TM_SPEC_Z], h->spec, 2LL * h->nxhp, h->ny, np, 2 * TCOLS, 1, bz);
    {   // the folded V_dd table, boxes along the last axis (rows 0 .. N/2; fmi_vrows)
        const int nl = h->p.ndim == 3 ? h->nz : h->ny;
        if (nl == 128 || nl == 256 || nl == 512) {
            if (h->p.ndim == 3) rc |= make_map((CUtensorMap*)h->tmap[TM_VDD], h->vdd, h->nxhp, h->nyf, h->nzf, TCOLS, 1, fmi_vrows(nl));
            else rc |= make_map((CUtensorMap*)h->tmap[TM_VDD], h->vdd, h->nxhp, h->nyf, 1, TCOLS, fmi_vrows(nl), 1);
        }
    }
    if (h->nx == 128 || h->nx == 256 || h->nx == 512) {
        // kernels_xwarp.cu: an x-line as NX/8 rows of 128 bytes (8 complex), a box = all rows of 2 (NX = 256, 512) or
        // 4 (NX = 128) lines, 16-byte units of a row rotated by the row index (SWIZZLE_128B)
        const int lpt = h->nx == 128 ? 4 : 2;
        rc |= make_map((CUtensorMap*)h->tmap[TM_PSI_XW], h->psi, 16, h->nx / 8, (long long)h->ny * np, 16, h->nx / 8, lpt, true);
    }
    return rc ? (int)cudaErrorInvalidValue : 0;
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
static TileGeom geom_of(const dbec_handle_s* h, int axis, bool sp, int z0, int nzs) {
    TileGeom tg;
    tg.rev = h->rev_next;
    tg.ystep = 1;
    tg.fold_pairs = 0;
    tg.pace_ns = 0; tg.pace_head = 0; tg.pace_head_ns = 0; tg.pace = nullptr;
    const int row_elems = sp ? h->nxhp : h->nx;          // a pass over the half spectrum or over psi
    tg.pol_ld = h->pol[sp ? POL_FFT_LD : POL_CN_LD];
    tg.pol_st = h->pol[sp ? POL_FFT_ST : POL_CN_ST];
    tg.axis = axis;
    tg.vfold = axis == 2 ? h->ny : 0;
    tg.vrows = fmi_vrows(axis == 1 ? h->ny : h->nz);
    tg.vnbox = fmi_vnbox(axis == 1 ? h->ny : h->nz);
    tg.ntiles_x = row_elems / TCOLS;
    const int n = axis == 1 ? h->ny : h->nz;
    tg.box_rows = box_rows_of(n);
    tg.nbox = n / tg.box_rows;
    if (axis == 1) { tg.ntiles = tg.ntiles_x * nzs; tg.outer0 = z0; }
    else { tg.ntiles = tg.ntiles_x * h->ny; tg.outer0 = 0; }
    return tg;
}

static int grid_of(const dbec_handle_s* h, int ntiles) { return ntiles < h->num_sms ? ntiles : h->num_sms; }

// Pacing of a streaming pass (tma_pipe.cuh: pace_wait).  tile_bytes: what one tile reads and writes; field_bytes:
// the field the pass streams.  The share of the field the previous pass left in L2 (about 0.8 of the cache, walked
// first thanks to the alternating tile order) is scheduled at pace_head_speed of the paced interval; a field that fits
// there is never paced.
PaceArgs dbec_pace_args(const dbec_handle_s* h, int ntiles, int grid, size_t tile_bytes, double field_bytes) {
    PaceArgs pa; pa.ns = 0; pa.head = 0; pa.head_ns = 0; pa.st = nullptr;
    if (h->pace_gbs <= 0.0 || grid < 1) return pa;
    const double head = 0.8 * (double)h->l2_bytes / field_bytes;
    if (head >= 1.0) return pa;
    const int per_cta = ntiles / grid;
    if (per_cta < 8) return pa;
    pa.ns = (int)((double)tile_bytes * grid / h->pace_gbs);
    if (pa.ns < 1) pa.ns = 1;
    pa.head = (int)(head * per_cta);
    pa.head_ns = (int)(h->pace_head_speed * pa.ns);
    pa.st = (PaceState*)(h->ticket + 16);          // 64 bytes into the ticket block
    return pa;
}
static void set_pace(const dbec_handle_s* h, TileGeom* tg, int grid, size_t tile_bytes, double field_bytes) {
    const PaceArgs pa = dbec_pace_args(h, tg->ntiles, grid, tile_bytes, field_bytes);
    tg->pace_ns = pa.ns; tg->pace_head = pa.head; tg->pace_head_ns = pa.head_ns; tg->pace = pa.st;
}

template <bool RT, int NCH, int NG, int NST, bool NORM, int TC = TCOLS> static int launch_cn_tma(dbec_handle_s* h, int axis, int z0, int nzs) {
    constexpr int GT = NCH * TC, STAGE = NCH * CN_L * TC * (int)sizeof(cd);
    TileGeom tg = geom_of(h, axis, false, z0, nzs);
    if (TC == 2 * TCOLS) { tg.ystep = 2; tg.ntiles = tg.ntiles_x * (h->ny / 2); }
    const int grid = grid_of(h, tg.ntiles);
    if (NORM && (grid > h->npartial || h->nb > 1)) return (int)cudaErrorInvalidValue;   // a CTA's tiles span members
    set_pace(h, &tg, grid, 2 * (size_t)STAGE, 16.0 * (double)h->P * h->nb);
    const size_t sm = 128 + (size_t)NST * STAGE + (size_t)NG * 2 * GT * sizeof(cd) + (3 * NST + 4) * sizeof(uint64_t) +
                      (3 * cn_tab_elems(NCH * CN_L) + 2 * NCH) * sizeof(typename CnCoef<RT>::type);
    auto k = k_cn_tma<RT, NCH, NG, NST, NORM, TC>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const CUtensorMap* map = (const CUtensorMap*)h->tmap[axis == 1 ? TM_PSI_Y : TC == 2 * TCOLS ? TM_PSI_Z2 : TM_PSI_Z];
    CK(launch_pdl(k, dim3(grid), dim3(NG * GT + 96), sm, h->stream, h->use_pdl, *map, make_cntab<RT>(h->ax[axis]), tg, h->partial,
                  h->ticket, h->scal, h->dV));
    h->launches++;
    return (int)cudaGetLastError();
}

template <bool RT, bool NORM> static int launch_cn_tma_n(dbec_handle_s* h, int axis, int z0, int nzs) {
    switch (h->ax[axis].n) {
        case 128:
            if (axis == 2 && dbec_zpair_tiles(h)) return launch_cn_tma<RT, 8, 3, 6, NORM, 2 * TCOLS>(h, axis, z0, nzs);    // 32 KiB tiles
            return launch_cn_tma<RT, 8, 4, 12, NORM>(h, axis, z0, nzs);     // 16 KiB tiles
        case 256:
            if (axis == 2 && dbec_zpair_tiles(h)) return launch_cn_tma<RT, 16, 1, 3, NORM, 2 * TCOLS>(h, axis, z0, nzs);   // 64 KiB tiles
            return launch_cn_tma<RT, 16, 3, 6, NORM>(h, axis, z0, nzs);     // 32 KiB tiles
        case 512: return launch_cn_tma<RT, 32, 1, 3, NORM>(h, axis, z0, nzs);     // 64 KiB tiles
        default: return (int)cudaErrorInvalidValue;
    }
}

// z sweeps on tiles of 8 columns x 2 rows of y: planes at least 2 MiB apart
int dbec_zpair_tiles(const dbec_handle_s* h) {
    return h->p.ndim == 3 && h->nb == 1 && h->ny % 2 == 0 && (long long)h->nx * h->ny * (long long)sizeof(cd) >= h->zpair_min_stride;
}

int dbec_tma_supported(const dbec_handle_s* h, int axis) {
    const int n = h->ax[axis].n;
    // batches: 2-D grids only (their planes stack along the tensor maps' outer coordinate); a batch of 3-D
    // grids runs its strided passes in the one-tile-per-block kernels
    if (h->nb > 1 && h->p.ndim == 3) return 0;
    return h->use_tma && (n == 128 || n == 256 || n == 512);
}

int dbec_launch_cn_tma(dbec_handle_s* h, int axis, int with_norm, int z0, int nzs) {
    if (h->p.time_mode == 1)
        return with_norm ? launch_cn_tma_n<true, true>(h, axis, z0, nzs) : launch_cn_tma_n<true, false>(h, axis, z0, nzs);
    return with_norm ? launch_cn_tma_n<false, true>(h, axis, z0, nzs) : launch_cn_tma_n<false, false>(h, axis, z0, nzs);
}

template <int N> struct PlanS;
template <> struct PlanS<128> { typedef FftPlan<8, 1, false> P; };
template <> struct PlanS<256> { typedef FftPlan<16, 1, false> P; };
template <> struct PlanS<512> { typedef FftPlan<16, 2, false> P; };

template <int N, int MODE, int NG, int NST> static int launch_fft_tma(dbec_handle_s* h, int axis, int z0, int nzs) {
    typedef typename PlanS<N>::P P;
    constexpr int GT = P::T * TCOLS;
    constexpr int STAGE = N * TCOLS * (int)sizeof(cd) + (MODE == 2 ? fmi_extra_bytes(N) : 0);
    TileGeom tg = geom_of(h, axis, true, z0, nzs);
    // (measured: the step 480.3 -> 478.7 us at 256^3, 1951.7 -> 1949.5 at 512 x 512 x 256)
    if (MODE == 2 && axis == 2 && h->ny % 2 == 0) tg.fold_pairs = h->ny;
    const int grid = grid_of(h, tg.ntiles);
    set_pace(h, &tg, grid, (size_t)STAGE + N * TCOLS * sizeof(cd), 16.0 * (double)h->SP * h->nb);
    const size_t sm = 128 + (size_t)NST * STAGE + (3 * NST + 4) * sizeof(uint64_t) + 2 * N * sizeof(cd);
    auto k = k_fft_tma<P, MODE, NG, NST>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const CUtensorMap* map = (const CUtensorMap*)h->tmap[axis == 1 ? TM_SPEC_Y : TM_SPEC_Z];
    const CUtensorMap* mv = (const CUtensorMap*)h->tmap[TM_VDD];
    CK(launch_pdl(k, dim3(grid), dim3(NG * GT + 96), sm, h->stream, h->use_pdl, *map, *mv, h->ax[axis].twA, h->ax[axis].twN, tg));
    h->launches++;
    return (int)cudaGetLastError();
}

template <int MODE> static int launch_fft_tma_n(dbec_handle_s* h, int axis, int z0, int nzs) {
    switch (h->ax[axis].n) {
        case 128: return launch_fft_tma<128, MODE, 4, (MODE == 2 ? 10 : 12)>(h, axis, z0, nzs);
        case 256: return launch_fft_tma<256, MODE, 2, (MODE == 2 ? 5 : 6)>(h, axis, z0, nzs);
        case 512: return launch_fft_tma<512, MODE, 1, (MODE == 2 ? 2 : 3)>(h, axis, z0, nzs);
        default: return (int)cudaErrorInvalidValue;
    }
}

int dbec_launch_fft_tma(dbec_handle_s* h, int axis, int mode, int z0, int nzs) {
    if (mode == 0) return launch_fft_tma_n<0>(h, axis, z0, nzs);
    if (mode == 1) return launch_fft_tma_n<1>(h, axis, z0, nzs);
    return launch_fft_tma_n<2>(h, axis, z0, nzs);
}
