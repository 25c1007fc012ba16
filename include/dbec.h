/* dbec.h — C ABI of the B200-native dipolar SSCN step (arxiv 1601.04640, "DBEC-GP-CUDA").
 *
 * One split-step semi-implicit Crank-Nicolson (SSCN) time step of the 2-D/3-D dipolar
 * Gross-Pitaevskii equation, in imaginary or real time ("Nature of problem",
 * "Solution method"), behind plain pointers and sizes.  Every step of the path runs in hand-written
 * sm_100a kernels inside libdbec.so; there is no CPU fallback and no library FFT.
 *
 * Problem (readings S1, S2, S3 of DESIGN.md; PAPER.md prints no formula):
 *     i dpsi/dt = [ -1/2 Lap + V + G |psi|^2 + D Phi_dd ] psi,   int |psi|^2 = 1,
 *     V = 1/2 (nu^2 x^2 + lambda^2 y^2 + kappa^2 z^2),
 *     Phi_dd = F^-1[ V_dd(k) F[|psi|^2] ],  V_dd(k) = 3 k_z^2/|k|^2 - 1  (3-D; 0 at k = 0);
 *     2-D: that kernel averaged over the frozen Gaussian direction of width d_perp (S21, S25).
 * The six programs of the paper are the parameter sets (ndim, plane, time_mode) =
 *     imag2dXY (2,0,0)  imag2dXZ (2,1,0)  imag3d (3,0,0)  real2dXY (2,0,1)  real2dXZ (2,1,1)  real3d (3,0,1).
 * One step (PAPER.md:67 function list; order = reading S10):
 *     calcpsidd2 (density -> FFT -> x V_dd -> inverse FFT), calcnu (psi *= exp(-c dt (V+G n+D Phi))),
 *     calclux, calcluy, calcluz (Crank-Nicolson tridiagonal solve on every grid line),
 *     calcnorm (imaginary time only).  c = 1 in imaginary time, i in real time.
 *
 * Layout of every field: x fastest, idx = ix + NX*(iy + NY*iz); psi is complex128 stored as
 * (re, im) pairs of IEEE doubles.  Grid coordinates x_i = (i - NX/2)*dx (reading S17).
 *
 * Ownership: the caller owns all device memory, including the workspace handed to dbec_create
 * (size from dbec_workspace_bytes, 256-byte aligned); the library owns only the small host-side
 * handle.  dbec_set_psi / dbec_get_psi copy, they never adopt the caller's buffer.
 *
 * Errors: every call returns 0 (DBEC_OK) or a negative code; nothing throws or aborts; NULL
 * arguments give DBEC_EINVAL.  All work is enqueued on the CUDA stream given to dbec_create.
 */
#ifndef DBEC_H
#define DBEC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DBEC_OK           0
#define DBEC_EINVAL      -1   /* NULL pointer, bad ndim / time_mode / spacing, nsteps < 0 ...        */
#define DBEC_ESIZE       -2   /* grid length not a supported FFT length (never silently adjusted,
                                 contrast PAPER.md:93); supported: 4..1024 with prime factors 2, 3,
                                 5, 7 only, NX even, NY*NZ even                                     */
#define DBEC_EWORKSPACE  -3   /* workspace NULL, misaligned or smaller than dbec_workspace_bytes    */
#define DBEC_ECUDA       -4   /* a CUDA call failed; dbec_last_cuda_error gives the CUDA code       */
#define DBEC_ENODEVICE   -5   /* no CUDA device / not an sm_100 device                              */
#define DBEC_ENOALLOC_SIZE -6 /* dbec_norm_noalloc: more than DBEC_NOALLOC_MAX_POINTS points         */

typedef struct dbec_handle_s* dbec_handle;

typedef struct {
    int32_t ndim;              /* 2 or 3                                                            */
    int32_t plane;             /* 2-D only: 0 = XY (dipoles along the frozen axis, reading S21);
                                  1 = XZ (dipoles IN the plane, the imag2dXZ / real2dXZ programs of
                                  PAPER.md:15, :119-131, :163-177, reading S25): the second grid axis
                                  (ny, dy, lambda) is then the polarisation axis z and y is frozen;
                                  must be 0 in 3-D                                                   */
    int32_t nx, ny, nz;        /* nz = 1 in 2-D                                                     */
    double  dx, dy, dz;        /* grid spacings (dz ignored in 2-D)                                 */
    double  dt;                /* time step                                                         */
    double  nu, lambda, kappa; /* trap anisotropies along x, y, z (reading S2)                      */
    double  G, D;              /* coefficients of |psi|^2 and of Phi_dd (reading S3)                */
    double  d_perp;            /* 2-D only: Gaussian width of the frozen direction (reading S21)    */
    double  cutoff;            /* 3-D only: spherical truncation radius of V_dd, 0 = none (S5)      */
    int32_t time_mode;         /* 0 = imaginary time, 1 = real time                                 */
} dbec_params;

/* calcmuen / calcrms; definitions in DESIGN.md "Observables" (readings S13-S16). */
typedef struct {
    double norm, mu, energy, rms_x, rms_y, rms_z, rms_r, density0, density_max;
} dbec_obs;

/* Bytes of device workspace dbec_create needs for these parameters (host call, no CUDA work). */
int dbec_workspace_bytes(const dbec_params* p, size_t* bytes);

/* Build a handle.  dev_workspace: DEVICE pointer, >= *bytes, 256-byte aligned, owned by the caller
 * and kept alive until dbec_destroy.  cuda_stream: a cudaStream_t (NULL = default stream).
 * Builds on the device the tables the paper's CPU initialises (`pot`, `potdd`)
 * and the Crank-Nicolson coefficients of each axis.  psi starts as all zeros. */
int dbec_create(const dbec_params* p, void* dev_workspace, size_t bytes, void* cuda_stream,
                dbec_handle* out);

/* Copy NX*NY*NZ complex128 values into the handle's psi.  psi_c128: HOST pointer if on_device == 0
 * (synchronous copy), DEVICE pointer otherwise (asynchronous on the handle's stream). */
int dbec_set_psi(dbec_handle h, const void* psi_c128, int on_device);

/* Copy psi out (same pointer rules), with the deferred imaginary-time norm factor applied. */
int dbec_get_psi(dbec_handle h, void* psi_c128, int on_device);

/* The same two copies for PINNED host buffers (cudaHostAlloc / cudaHostRegister), without the host synchronisation:
 * the copy is enqueued on the handle's stream and the call returns at once, so the transfers of one handle overlap
 * the steps and the opposite-direction transfers of another (a few handles on streams of their own taking turns
 * keep both directions of the host link busy — how bench.py's end-to-end leg feeds the GPU).  The buffer must stay valid and untouched
 * until the stream has passed the copy: dbec_synchronize, or the caller's own event on that stream.  With pageable
 * memory CUDA stages the copy and the call may block; the result is the same.  Only the state handed over
 * changes hands ("only wave function array is returned"); nothing else crosses the link. */
int dbec_set_psi_async(dbec_handle h, const void* psi_c128_host);
int dbec_get_psi_async(dbec_handle h, void* psi_c128_host);

/* Block the calling host thread until everything enqueued on the handle's stream has finished. */
int dbec_synchronize(dbec_handle h);

/* Change G and D (quench, reading S18).  Takes effect from the next step; ends a running ramp.  On a batch
 * handle every member gets the same pair. */
int dbec_set_coupling(dbec_handle h, double G, double D);

/* NSTP ramp of the nonlinearity ("NSTP"; reading S26): the k-th dbec_step after this
 * call (k = 1..nstp) runs with G0 + (G1 - G0) k/nstp and D0 + (D1 - D0) k/nstp, every later one with (G1, D1).
 * nstp = 0: (G1, D1) at once — the paper's NSTP = 0 restart is then dbec_set_psi of a stored state, e.g. the
 * device buffer dbec_get_psi filled from an imaginary-time handle.  The schedule lives in device memory, so the
 * CUDA graph of a step sees it; dbec_observables / dbec_phi_dd do not advance it. */
int dbec_set_ramp(dbec_handle h, int nstp, double G0, double D0, double G1, double D1);

/* nsteps SSCN steps, asynchronous on the handle's stream, no host sync.  3-D grids of up
 * to 65536 points per batch member (131072 when every length is 16, 32 or 64) run all nsteps steps in ONE launch by
 * thread-block clusters, one member per cluster at a time (PAPER.md:79 on launch overhead; environment
 * DBEC_CLUSTER=0 at dbec_create switches that off); larger grids replay a CUDA graph of the step's seven launches. */
int dbec_step(dbec_handle h, int nsteps);

/* calcmuen + calcrms on the current psi.  host_out: HOST pointer.  Synchronises
 * the stream.  In 2-D rms_x / rms_y are those of the two grid axes, rms_z = 0. */
int dbec_observables(dbec_handle h, dbec_obs* host_out);

int dbec_destroy(dbec_handle h);

/* ---- batched handles: nbatch independent simulations with the same parameters advance in the
 * same kernel launches — the only way grids as small as 32^3 or 512^2, whose single step is bound by launch
 * latency ("launching of all required kernels would create a sizeable overhead"), fill the GPU.
 * Every field is member-major: dbec_set_psi / dbec_get_psi move nbatch * NX*NY*NZ values; dbec_step,
 * dbec_set_ramp, dbec_set_coupling, dbec_normalize, dbec_cn_sweep, dbec_nonlinear, dbec_phi_dd act on all
 * members.  1 <= nbatch <= 65536.  dbec_create == dbec_create_batch with nbatch = 1. ---- */
int dbec_workspace_bytes_batch(const dbec_params* p, int nbatch, size_t* bytes);
int dbec_create_batch(const dbec_params* p, int nbatch, void* dev_workspace, size_t bytes, void* cuda_stream,
                      dbec_handle* out);
int dbec_batch_size(dbec_handle h, int* nbatch);
/* Per-member couplings (parameter scans): G, D HOST arrays of nbatch values. */
int dbec_set_coupling_batch(dbec_handle h, const double* G, const double* D);
/* host_out: HOST array of nbatch records.  dbec_observables itself returns DBEC_EINVAL on a handle with
 * more than one member. */
int dbec_observables_batch(dbec_handle h, dbec_obs* host_out);

/* ---- integrated densities (reading S27; the lineage's density output): |psi|^2 of batch member
 * `member` summed over the other axes times their spacings.  out: HOST (synchronises) or DEVICE pointer. ----
 * 1-D along `axis` (0 x, 1 y, 2 z; < ndim): N_axis doubles. */
int dbec_density_1d(dbec_handle h, int member, int axis, double* out, int on_device);
/* 2-D, 3-D grids only, integrated over `axis_integrated`: the two remaining axes, the lower one fastest
 * (2: [NY][NX], 1: [NZ][NX], 0: [NZ][NY]). */
int dbec_density_2d(dbec_handle h, int member, int axis_integrated, double* out, int on_device);

const char* dbec_strerror(int code);
/* CUDA error code behind this handle's last DBEC_ECUDA (0 if none).  h == NULL: the CUDA error behind the
 * calling thread's last failed dbec_create, which leaves no handle to ask. */
int dbec_last_cuda_error(dbec_handle h);

/* ---- single parts of the step, exported so that each can be checked on its own ---- */

/* calcpsidd2 alone: Phi_dd of the current psi into phi_f64, NX*NY*NZ doubles,
 * DEVICE pointer, asynchronous. */
int dbec_phi_dd(dbec_handle h, void* phi_f64_dev);

/* calclux / calcluy / calcluz alone: one Crank-Nicolson sweep along axis 0, 1 or 2
 * applied to psi in place, asynchronous. */
int dbec_cn_sweep(dbec_handle h, int axis);

/* calcnu alone: psi *= exp(-c dt (V + G|psi|^2 + D Phi_dd)) with Phi_dd of the
 * current psi, no Crank-Nicolson sweep, asynchronous. */
int dbec_nonlinear(dbec_handle h);

/* calcnorm alone: psi <- psi / sqrt(dV sum |psi|^2), asynchronous.  In imaginary time the
 * factor is kept deferred (applied by every consumer); in real time, where no step ever renormalises, it is
 * applied to the stored field at once. */
int dbec_normalize(dbec_handle h);

/* Number of kernel launches the library has enqueued on this handle since creation. */
int dbec_launch_count(dbec_handle h, long long* launches);

/* Measurement aid (bench.py's roofline leg): nsteps steps with plain launches and a CUDA event pair
 * around every kernel.  ms_per_slot: HOST pointer to DBEC_KERNEL_SLOTS doubles receiving the total
 * milliseconds spent in each kernel slot over the nsteps steps; launches_per_slot: HOST pointer to
 * DBEC_KERNEL_SLOTS counts.  Synchronises the stream.  Slot names from dbec_kernel_name. */
#define DBEC_KERNEL_SLOTS 9
int dbec_step_profile(dbec_handle h, int nsteps, double* ms_per_slot, long long* launches_per_slot);
const char* dbec_kernel_name(int slot);
/* Name of the __global__ function that serves pass `slot` on this handle ("" if the pass is not part
 * of this handle's dbec_step): grid lines of 128..512 points run in the persistent TMA-fed kernels,
 * shorter ones in the one-tile-per-block kernels; on a small grid the only slot is the last one,
 * "sscn_step<cluster>" (k_small_step). */
const char* dbec_pass_kernel(dbec_handle h, int slot);

/* calcnorm for callers that may not allocate (CUDA graph capture, serving loops): the norm
 * integral dV * sum |psi|^2 of npoints complex128 values, written to *norm_dev.  No handle, no workspace: the
 * block partial sums live in a device array of DBEC_NOALLOC_SCRATCH_BYTES that is part of the library image
 * (held by every GPU that loads the library, until exit); the call issues no cudaMalloc / cudaFree.
 *   psi_c128_dev, norm_dev: DEVICE pointers (inputs and outputs stay the caller's); cuda_stream: a cudaStream_t
 *   (NULL = the default stream).  Asynchronous on that stream; one memset node and one kernel.
 *   npoints > DBEC_NOALLOC_MAX_POINTS -> DBEC_ENOALLOC_SIZE;  NULL pointer, npoints < 1, dV <= 0 -> DBEC_EINVAL;
 *   a failed CUDA call -> DBEC_ECUDA with the CUDA code in dbec_noalloc_last_cuda_error() (per host thread).
 * All calls on a device share the one array: calls that overlap on the GPU (different streams, several host
 * threads) race; put them on one stream or serialise them.  Same fixed-order sum on every GPU. */
#define DBEC_NOALLOC_MAX_POINTS    134217728LL     /* 2^27 */
#define DBEC_NOALLOC_SCRATCH_BYTES 262400          /* 32768 partial sums + a 256-byte ticket */
int dbec_norm_noalloc(const void* psi_c128_dev, long long npoints, double dV, double* norm_dev, void* cuda_stream);
int dbec_noalloc_last_cuda_error(void);

int dbec_version(void);
/* "DBEC_BUILD_ID=<hash of the sources this library was built from>" (paper_1601_04640_b200/build.py). */
const char* dbec_build_id(void);

#ifdef __cplusplus
}
#endif
#endif /* DBEC_H */
