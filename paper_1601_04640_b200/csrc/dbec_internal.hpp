// dbec_internal.hpp — what the translation units of libdbec.so share: the host-side handle and the
// launcher prototypes.  Product path only; nothing here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/dbec.h"
#include "cplx.cuh"

#define DBEC_MAX_N 1024         // longest supported grid line
#define DBEC_MAX_KERNELS 9      // kernel slots of one step (dbec_step_profile); the last one is the one-launch small-grid step
#define DBEC_SPEC_COLS 8        // columns per tile of the strided FFT passes (8 x 16 B = one 128 B line)
#define DBEC_TMAP_BYTES 128     // sizeof(CUtensorMap)

// Access sites with an L2 eviction hint: loads / stores of psi in k_cn_tma, of psi and of the spectrum in
// k_xline_nonlin, of psi and the spectrum in k_xline_density, of the spectrum in k_fft_tma.
enum { POL_CN_LD = 0, POL_CN_ST, POL_NL_LD, POL_NL_ST, POL_NL_SPEC, POL_D_PSI, POL_D_SPEC, POL_FFT_LD, POL_FFT_ST, POL_COUNT };

// Tensor maps of the handle (kernels_tma.cu): field x direction of the box rows.
// TM_PSI_XW: psi as [line][NX/8][8 complex] with the 128-byte swizzle (kernels_xwarp.cu).
// TM_VDD: the folded V_dd table, boxes along the last axis of the grid.
// TM_PSI_Z2: psi with boxes of 8 columns x 2 rows of y x N rows of z (k_cn_tma with TC = 16).
enum { TM_PSI_Y = 0, TM_PSI_Z, TM_SPEC_Y, TM_SPEC_Z, TM_VDD, TM_PSI_XW, TM_PSI_Z2, TM_COUNT };

// Device scalars every kernel reads (so that a captured CUDA graph never bakes them in), one block of
// SC_COUNT doubles per batch member (dbec_create_batch; a plain handle has one member).
//   [0] s      deferred norm factor: true psi = s * stored psi (calcnorm; 1 in real time)
//   [1] s^2
//   [2] G      coefficient of |psi|^2 used by the current step   (dbec_set_coupling / the ramp below)
//   [3] D      coefficient of Phi_dd
//   [4..7]     G0, D0, G1, D1 of the NSTP ramp (dbec_set_ramp, reading S26)
//   [8], [9]   ramp steps begun so far, ramp length (as doubles); no ramp: both 0
enum { SC_S = 0, SC_S2 = 1, SC_G = 2, SC_D = 3, SC_G0 = 4, SC_D0 = 5, SC_G1 = 6, SC_D1 = 7, SC_RK = 8, SC_RN = 9, SC_COUNT = 16 };

#if defined(__CUDACC__)
// Reading S26 ("NSTP"): the k-th step after dbec_set_ramp (k = 1..n) runs with
// G0 + (G1 - G0) k/n and D0 + (D1 - D0) k/n.  Called by ONE thread per member in the first kernel of a step
// (the density pass, which reads neither G nor D); the nonlinear kernel later in the stream sees the result.
__device__ __forceinline__ void ramp_advance(double* __restrict__ sc) {
    const double k = sc[SC_RK], n = sc[SC_RN];
    if (k < n) {
        const double k1 = k + 1.0, f = k1 / n;
        sc[SC_RK] = k1;
        sc[SC_G] = sc[SC_G0] + (sc[SC_G1] - sc[SC_G0]) * f;
        sc[SC_D] = sc[SC_D0] + (sc[SC_D1] - sc[SC_D0]) * f;
    }
}
#endif

// Pacing of the streaming passes (tma_pipe.cuh: pace_wait).  PaceState: one word per handle in the ticket block.
struct PaceState { unsigned long long lag; unsigned int exits; unsigned int pad; };
struct PaceArgs {
    int ns;             // interval at which a loader issues its tiles, 0 = no pacing
    int head, head_ns;  // the first `head` tiles of a CTA (they come out of L2) at this shorter interval
    PaceState* st;
};

// Per-axis tables on the device.
struct AxisTables {
    int n;                  // points along the axis
    const cd* twA;          // stage-1 FFT twiddles, order [k1][m]           (n entries)
    const cd* twN;          // exp(-2 pi i j / n)                              (n entries)
    const double* vtrap;    // 1/2 omega^2 x_i^2                               (n entries)
    const double* x2;       // x_i^2                                           (n entries)
    // Crank-Nicolson tables (cn_chunk.cuh): real in imaginary time, complex in real time; stored as
    // complex in both cases, the imaginary-time kernels read the real parts only through *_re.
    // pfe[c] = PF at the last point of chunk c, pbs[c] = PB at the first point of chunk c.
    const cd* h;  const cd* pf;  const cd* pb;  const cd* pfe;  const cd* pbs;
    const double* h_re; const double* pf_re; const double* pb_re; const double* pfe_re; const double* pbs_re;
    cd kap;                 // (1 - 2a)/a
    // the same tables for chunks of 8 points (kernels_xwarp.cu; built for the x axis only) and the number of
    // carry terms that are above 2^-73 of the leading one (0: tables not built)
    const cd* pf8; const cd* pb8; const cd* pfe8; const cd* pbs8;
    const double* pf8_re; const double* pb8_re; const double* pfe8_re; const double* pbs8_re;
    int K8;
    int K16;                // the same count for the chunks of 16 points (kernels_gen.cu)
};

struct dbec_handle_s {
    dbec_params p;
    cudaStream_t stream;
    int last_cuda;
    long long launches;
    // geometry
    int nx, ny, nz, nxhp;           // nxhp = padded half-spectrum row length (multiple of DBEC_SPEC_COLS)
    long long P;                    // nx*ny*nz   (per batch member)
    long long SP;                   // nz*ny*nxhp (per batch member)
    double dV;
    // batch (dbec_create_batch): nb independent members with the same parameters; every field
    // below holds the members back to back (member-major), the V_dd table and the axis tables are shared
    int nb;
    int nplanes;                    // nz * nb: xy planes in psi / spec (a batch of 2-D grids is a stack of planes)
    // device memory (all inside the caller's workspace)
    cd* psi;                        // [nz][ny][nx]
    cd* spec;                       // [nz][ny][nxhp] half spectrum of the density
    // V_dd(k)/P folded by its even symmetry in k_y and k_z (V_dd(k) depends on the squares of the wavenumbers and
    // index m and N - m carry +-k: bitwise the same value): [nzf][nyf][nxhp], nyf = ny/2 + 1, nzf = nz/2 + 1 (1 in
    // 2-D).  A quarter of the full table (17 MiB instead of 68 MiB at 256^3).
    double* vdd;
    int nyf, nzf;
    double* phi;                    // [nz][ny][nx] Phi_dd (observables / dbec_phi_dd only)
    double* scal;                   // nb x SC_COUNT doubles
    double* partial;                // reduction partials
    unsigned int* ticket;           // last-block tickets
    double* obs_dev;                // nb x 16 doubles
    AxisTables ax[3];
    // axes whose length is not one of the powers of two 16..512 run in the run-time-length kernels of
    // kernels_gen.cu: gen[axis] = 1, radices of the Stockham passes in gfac[axis][0..gnfac)
    int gen[3], gnfac[3], gfac[3][12];
    int npartial;
    // CUDA graph of one step
    cudaGraphExec_t graph_exec;
    int launches_per_step;
    // per-kernel timing (dbec_step_profile): event pairs around every launch of a step
    int prof_on, prof_n;
    cudaEvent_t prof_ev[2 * DBEC_MAX_KERNELS];
    int prof_slot[DBEC_MAX_KERNELS];
    int use_graph;                  // env DBEC_GRAPH (default 1): replay one captured step per dbec_step iteration
    int fuse_cnx;                   // env DBEC_FUSE_CNX (default 1): x sweep inside the nonlinear kernel
    int use_tma;                    // 1: persistent TMA-fed kernels for lines of 128..512 points
    int num_sms;
    int use_cluster;                // CTAs per cluster of the one-launch small-grid step, 0 = not used (dbec_small_choose;
                                    // env DBEC_CLUSTER = 0 / 1 / 2 / 4 / 8 / 16 overrides the choice)
    int use_small;                  // 1: dbec_step runs k_small_step (use_cluster > 0)
    int small_max_clusters;         // clusters of k_small_step that can be resident at once (0: not asked yet)
    int use_small_p2;               // 1: the small-grid step runs in k_small_p2 (kernels_small_p2.cu: compiled power-of-two shapes)
    double pace_gbs;                // bandwidth the streaming passes are paced to, GB/s (tma_pipe.cuh: pace_wait); 0 = off
    long long l2_bytes;             // L2 cache size of the device
    double pace_head_speed;         // time per tile of the L2-resident head of a pass relative to the paced time
    long long zpair_min_stride;     // z sweeps pair two rows of y per tile when the xy plane is at least this many bytes
    int use_pdl;                    // 1: programmatic dependent launch of every kernel of a step
    int rev_next;                   // the next persistent launch walks its tiles last to first (L2 reuse across passes)
    int use_rev;                    // 1: consecutive plane-ordered passes walk their tiles in opposite directions
    // L2 eviction policy code of every bulk / TMA access site (tma_pipe.cuh: l2_policy_code)
    float pol[POL_COUNT];
    alignas(64) unsigned char tmap[TM_COUNT][DBEC_TMAP_BYTES];
};

// ---- launchers (each returns a cudaError_t as int; all asynchronous on h->stream) ----
// advance: 1 in a step (the density pass also moves the NSTP ramp on), 0 for observables / dbec_phi_dd
int dbec_launch_density_fftx(dbec_handle_s* h, int advance);   // a1, x axis: psi -> half spectrum
int dbec_launch_fft_strided(dbec_handle_s* h, int axis, int mode);   // a1/a3 along y or z; mode 0 forward, 1 inverse,
                                                           // 2 forward * V_dd(k)/P * inverse (a2 fused)
int dbec_launch_nonlinear(dbec_handle_s* h, int fuse_cnx); // a3 (x, C2R) + a4 [+ a5]
int dbec_launch_phi_out(dbec_handle_s* h, double* phi);    // a3 writing Phi_dd only (all members)
int dbec_launch_cn(dbec_handle_s* h, int axis, int with_norm);   // a5..a7 (+ a8 partial sums and factor)
int dbec_launch_normalize(dbec_handle_s* h);               // a8 alone (applies any deferred factor first)
int dbec_launch_norm_only(dbec_handle_s* h);               // a8 on a stored field with s = 1 (batched persistent sweeps)
int dbec_launch_apply_scale(dbec_handle_s* h);             // psi <- s psi, s <- 1
int dbec_launch_reset_scale(dbec_handle_s* h);             // s <- 1
int dbec_launch_observables(dbec_handle_s* h);             // a9 (expects h->phi filled), every member
int dbec_launch_density_2d(dbec_handle_s* h, int member, int axis, double* out);   // reading S27 (3-D grids)
int dbec_launch_density_1d(dbec_handle_s* h, int member, int axis, double* out, double* scratch);
int dbec_launch_build_vdd(dbec_handle_s* h);               // potdd table
// run-time line lengths 2^a 3^b 5^c 7^d (kernels_gen.cu)
int dbec_gen_factor(int n, int* fac);
int dbec_launch_gen_density_fftx(dbec_handle_s* h, int advance);
int dbec_launch_gen_fft(dbec_handle_s* h, int axis, int mode);
int dbec_launch_gen_nonlinear(dbec_handle_s* h);                // a3 (x) + a4, no sweep
int dbec_launch_gen_phi_out(dbec_handle_s* h, double* phi);
int dbec_launch_gen_cn(dbec_handle_s* h, int axis, int with_norm);
// persistent TMA-fed versions of the strided passes (kernels_tma.cu); z0, nzs: slab of planes (y passes)
int dbec_make_tensor_maps(dbec_handle_s* h);
int dbec_tma_supported(const dbec_handle_s* h, int axis);
int dbec_zpair_tiles(const dbec_handle_s* h);
// pacing of a launch of `grid` CTAs over `ntiles` tiles moving tile_bytes each while streaming a field of field_bytes
PaceArgs dbec_pace_args(const dbec_handle_s* h, int ntiles, int grid, size_t tile_bytes, double field_bytes);
int dbec_launch_fft_tma(dbec_handle_s* h, int axis, int mode, int z0, int nzs);
int dbec_launch_cn_tma(dbec_handle_s* h, int axis, int with_norm, int z0, int nzs);
// persistent bulk-copy-fed versions of the x passes (kernels_xline.cu)
int dbec_xline_supported(const dbec_handle_s* h);
int dbec_launch_xline_nonlin(dbec_handle_s* h, int z0, int nzs);          // a3 (x) + a4 + a5
int dbec_launch_xline_density(dbec_handle_s* h, int z0, int nzs, int advance);   // a1 (x)
// the whole step of a small grid in one launch by one thread-block cluster (kernels_small.cu)
int dbec_small_choose(dbec_handle_s* h, int request);     // CTAs per cluster (0: multi-launch path); request < 0: auto
int dbec_launch_small_step(dbec_handle_s* h, int nsteps);
int dbec_small_p2_choose(dbec_handle_s* h, int request);  // CTAs per cluster when k_small_p2 serves this handle, else 0 (sets small_max_clusters)
int dbec_launch_small_p2(dbec_handle_s* h, int nsteps);
// one warp per line pair (kernels_xwarp.cu): a3 (x) + a4 + a5 for lines of 128 / 256 points
int dbec_xwarp_supported(const dbec_handle_s* h);
int dbec_launch_xwarp_nonlin(dbec_handle_s* h);
