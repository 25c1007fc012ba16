// dbec_api.cu — the C ABI of include/dbec.h: parameter checks, workspace layout, table set-up, the
// order of the kernels inside one SSCN step (reading S10: calcpsidd2, calcnu, calclux, calcluy,
// calcluz, calcnorm — PAPER.md:67) and its CUDA graph.  No arithmetic of the method lives here.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <cmath>
#include <new>
#include <vector>
#include "dbec_internal.hpp"
#include "cn_chunk.cuh"
#include "host_tables.hpp"

#define DBEC_VERSION 200
#define DBEC_MAX_BATCH 65536

// Powers of two 16..512 run in the register-resident kernels, every other length 4..1024 with prime factors
// 2, 3, 5, 7 only in the run-time-length kernels (kernels_gen.cu).
static bool len_pow2_fast(int n) { return n == 16 || n == 32 || n == 64 || n == 128 || n == 256 || n == 512; }
static bool fft_len_ok(int n) {
    int fac[12];
    return n >= 4 && n <= DBEC_MAX_N && dbec_gen_factor(n, fac) > 0;
}

static int check_params(const dbec_params* p) {
    if (!p) return DBEC_EINVAL;
    if (p->ndim != 2 && p->ndim != 3) return DBEC_EINVAL;
    if (p->plane != 0 && !(p->ndim == 2 && p->plane == 1)) return DBEC_EINVAL;
    if (p->time_mode != 0 && p->time_mode != 1) return DBEC_EINVAL;
    if (!(p->dx > 0.0) || !(p->dy > 0.0) || !(p->dt > 0.0)) return DBEC_EINVAL;
    if (p->ndim == 3 && !(p->dz > 0.0)) return DBEC_EINVAL;
    if (p->ndim == 2 && !(p->d_perp > 0.0)) return DBEC_EINVAL;
    if (p->cutoff < 0.0) return DBEC_EINVAL;
    if (p->nx < 1 || p->ny < 1 || p->nz < 1) return DBEC_EINVAL;
    if (p->ndim == 2 && p->nz != 1) return DBEC_EINVAL;
    if (!fft_len_ok(p->nx) || !fft_len_ok(p->ny)) return DBEC_ESIZE;
    if (p->ndim == 3 && !fft_len_ok(p->nz)) return DBEC_ESIZE;
    // two real x-lines ride one complex transform: the lines pair up, and NX/2 is the Nyquist index
    if (p->nx % 2 || ((long long)p->ny * p->nz) % 2) return DBEC_ESIZE;
    return DBEC_OK;
}

// ---- workspace layout: one pass computes the offsets, used by both sizing and create ----
struct Layout {
    size_t psi, spec, vdd, phi, scal, partial, ticket, obs, tables, total;
    size_t tab_bytes, npartial;
};
static size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }

static size_t axis_table_bytes(int n_) {
    const int n = (n_ + 15) / 16 * 16;          // tables are zero-padded to whole Crank-Nicolson chunks
    // twA, twN (cd n each); vtrap, x2 (double n each); h, pf, pb (cd n each) + pfe, pbs (cd 32 each);
    // the same five as doubles; pf, pb for chunks of 8 (cd n each) + their pfe, pbs (cd 128 each), and as doubles
    size_t b = 0;
    b += up256(sizeof(cd) * n) * 2;
    b += up256(sizeof(double) * n) * 2;
    b += up256(sizeof(cd) * n) * 3 + up256(sizeof(cd) * 64) * 2;
    b += up256(sizeof(double) * n) * 3 + up256(sizeof(double) * 64) * 2;
    b += up256(sizeof(cd) * n) * 2 + up256(sizeof(cd) * 128) * 2;
    b += up256(sizeof(double) * n) * 2 + up256(sizeof(double) * 128) * 2;
    return b;
}

// Carry terms of the chunked Thomas solve that matter in fp64: the carry into a chunk is
// e[c-1] + f[c-1] (e[c-2] + f[c-2] (...)) with |f| = product of L consecutive |h_j| < 1; the q-th term is below
// fmax^(q-1) of the first.  Smallest K with fmax^K < 2^-73 (then every dropped term is below a quarter ulp of
// the sum even if the e's differ by three orders of magnitude), at most nchunks - 1.
static int carry_terms(const std::vector<dbec_host::zc>& f, int nchunks) {
    double fmax = 0.0;
    for (int c = 0; c < nchunks; ++c) fmax = std::max(fmax, std::abs(f[c]));
    if (nchunks <= 1 || fmax == 0.0) return 1;
    if (fmax >= 1.0) return nchunks - 1;
    const int k = (int)std::ceil(-73.0 * std::log(2.0) / std::log(fmax));
    return std::max(1, std::min(k, nchunks - 1));
}

// Reduction partials: one per block of the last Crank-Nicolson sweep (<= one per 256 points), ten per block
// of the observables pass.
static size_t npartial_of(size_t P, size_t nb, size_t last_sweep_columns = 0) {
    // last_sweep_columns: lines of the last sweep per member when it runs in kernels_gen.cu (one block per 8)
    size_t n = 32768, a = nb * P / 256 + nb, b = nb * 10 * 8, c = nb * (last_sweep_columns / 8 + 1);
    if (a > n) n = a;
    if (c > n) n = c;
    if (b > n) n = b;
    return n;
}

static void make_layout(const dbec_params* p, int nbatch, Layout* L) {
    const size_t nx = p->nx, ny = p->ny, nz = p->nz, nb = nbatch;
    const size_t nxhp = ((nx / 2 + 1) + DBEC_SPEC_COLS - 1) / DBEC_SPEC_COLS * DBEC_SPEC_COLS;
    const size_t P = nx * ny * nz, SP = nz * ny * nxhp;
    size_t o = 0;
    L->psi = o;     o += up256(nb * P * sizeof(cd));
    L->spec = o;    o += up256(nb * SP * sizeof(cd));
    L->vdd = o;     o += up256((nz / 2 + 1) * (ny / 2 + 1) * nxhp * sizeof(double));      // folded (dbec_internal.hpp)
    L->phi = o;     o += up256(nb * P * sizeof(double));
    L->scal = o;    o += up256(nb * SC_COUNT * sizeof(double));
    L->npartial = npartial_of(P, nb, p->ndim == 3 ? nx * ny : nx);
    L->partial = o; o += up256(L->npartial * sizeof(double));
    L->ticket = o;  o += 256;
    L->obs = o;     o += up256(nb * 16 * sizeof(double));
    L->tables = o;
    L->tab_bytes = axis_table_bytes(p->nx) + axis_table_bytes(p->ny) + axis_table_bytes(p->nz);
    o += L->tab_bytes;
    L->total = o;
}

static thread_local int create_cuda_error = 0;     // CUDA error of this thread's last failed dbec_create

static int cuda_fail(dbec_handle h, cudaError_t e) {
    if (h) h->last_cuda = (int)e;
    return DBEC_ECUDA;
}
#define CU(h, x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return cuda_fail(h, e_); } while (0)
#define LAUNCH(h, x) do { int rc_ = (x); if (rc_) return cuda_fail(h, (cudaError_t)rc_); } while (0)

// Upload one axis' tables; returns bytes consumed.
static int upload_axis(dbec_handle h, int axis, int n, double d, double omega, char* dev, size_t* used) {
    using namespace dbec_host;
    AxisTables& A = h->ax[axis];
    A.n = n;
    std::vector<zc> twN, twA, hh, pf, pb;
    std::vector<double> vtrap(n), x2(n);
    if (n >= 2) make_twN(n, twN); else twN.assign(1, zc(1.0, 0.0));
    if (len_pow2_fast(n)) make_twA(n, twN, twA); else twA = twN;
    for (int i = 0; i < n; ++i) {
        const double x = (double)(i - n / 2) * d;           // reading S17
        x2[i] = (n > 1) ? x * x : 0.0;
        vtrap[i] = (n > 1) ? 0.5 * omega * omega * x * x : 0.0;
    }
    const double ar = h->p.dt / (4.0 * d * d);              // a = c dt / (4 h^2), c = 1 or i
    const zc a = h->p.time_mode == 0 ? zc(ar, 0.0) : zc(0.0, ar);
    // any n >= 3; padded with zeros to whole chunks of CN_L points (kernels_gen.cu reads whole chunks: a padded
    // point has h = 0, solves to 0 and feeds nothing back)
    const int npad = (n + CN_L - 1) / CN_L * CN_L;
    if (n >= 3) make_cn(n, CN_L, a, hh, pf, pb);
    hh.resize(npad, zc(0, 0)); pf.resize(npad, zc(0, 0)); pb.resize(npad, zc(0, 0));
    std::vector<zc> pfe(64, zc(0, 0)), pbs(64, zc(0, 0));
    for (int c = 0; c < npad / CN_L; ++c) { pfe[c] = pf[c * CN_L + CN_L - 1]; pbs[c] = pb[c * CN_L]; }
    const zc kap = (1.0 - 2.0 * a) / a;
    A.kap = cmake(kap.real(), kap.imag());

    size_t o = 0;
    auto put = [&](const void* src, size_t bytes, const void** slot) -> cudaError_t {
        *slot = dev + o;
        cudaError_t e = cudaMemcpyAsync(dev + o, src, bytes, cudaMemcpyHostToDevice, h->stream);
        o += up256(bytes);
        return e;
    };
    auto re = [](const std::vector<zc>& v) { std::vector<double> r(v.size()); for (size_t i = 0; i < v.size(); ++i) r[i] = v[i].real(); return r; };
    std::vector<double> h_re = re(hh), pf_re = re(pf), pb_re = re(pb), pfe_re = re(pfe), pbs_re = re(pbs);
    CU(h, put(twA.data(), sizeof(zc) * n, (const void**)&A.twA));
    CU(h, put(twN.data(), sizeof(zc) * n, (const void**)&A.twN));
    CU(h, put(vtrap.data(), sizeof(double) * n, (const void**)&A.vtrap));
    CU(h, put(x2.data(), sizeof(double) * n, (const void**)&A.x2));
    CU(h, put(hh.data(), sizeof(zc) * npad, (const void**)&A.h));
    CU(h, put(pf.data(), sizeof(zc) * npad, (const void**)&A.pf));
    CU(h, put(pb.data(), sizeof(zc) * npad, (const void**)&A.pb));
    CU(h, put(pfe.data(), sizeof(zc) * 64, (const void**)&A.pfe));
    CU(h, put(pbs.data(), sizeof(zc) * 64, (const void**)&A.pbs));
    CU(h, put(h_re.data(), sizeof(double) * npad, (const void**)&A.h_re));
    CU(h, put(pf_re.data(), sizeof(double) * npad, (const void**)&A.pf_re));
    CU(h, put(pb_re.data(), sizeof(double) * npad, (const void**)&A.pb_re));
    CU(h, put(pfe_re.data(), sizeof(double) * 64, (const void**)&A.pfe_re));
    CU(h, put(pbs_re.data(), sizeof(double) * 64, (const void**)&A.pbs_re));
    A.K8 = 0;
    A.K16 = std::max(1, std::max(carry_terms(pfe, npad / CN_L), carry_terms(pbs, npad / CN_L)));
    if (n >= 3) {
        // the same tables for chunks of 8 points: the x axis of kernels_xwarp.cu (one 128-byte row of psi per lane) and
        // every axis of kernels_gen.cu (half the registers per thread, twice the threads per line); padded with zeros
        // to whole chunks like the tables above
        const int npad8 = (n + 7) / 8 * 8;
        std::vector<zc> h8, pf8, pb8, pfe8(128, zc(0, 0)), pbs8(128, zc(0, 0));
        make_cn(n, 8, a, h8, pf8, pb8);
        pf8.resize(npad8, zc(0, 0)); pb8.resize(npad8, zc(0, 0));
        for (int c = 0; c < npad8 / 8; ++c) { pfe8[c] = pf8[c * 8 + 7]; pbs8[c] = pb8[c * 8]; }
        std::vector<double> pf8_re = re(pf8), pb8_re = re(pb8), pfe8_re = re(pfe8), pbs8_re = re(pbs8);
        CU(h, put(pf8.data(), sizeof(zc) * npad8, (const void**)&A.pf8));
        CU(h, put(pb8.data(), sizeof(zc) * npad8, (const void**)&A.pb8));
        CU(h, put(pfe8.data(), sizeof(zc) * 128, (const void**)&A.pfe8));
        CU(h, put(pbs8.data(), sizeof(zc) * 128, (const void**)&A.pbs8));
        CU(h, put(pf8_re.data(), sizeof(double) * npad8, (const void**)&A.pf8_re));
        CU(h, put(pb8_re.data(), sizeof(double) * npad8, (const void**)&A.pb8_re));
        CU(h, put(pfe8_re.data(), sizeof(double) * 128, (const void**)&A.pfe8_re));
        CU(h, put(pbs8_re.data(), sizeof(double) * 128, (const void**)&A.pbs8_re));
        A.K8 = std::max(1, std::max(carry_terms(pfe8, npad8 / 8), carry_terms(pbs8, npad8 / 8)));
        CU(h, cudaStreamSynchronize(h->stream));          // the host vectors of this block go out of scope
    }
    // the host vectors must outlive the asynchronous copies from pageable memory: those copies are
    // staged synchronously by the runtime, but be explicit
    CU(h, cudaStreamSynchronize(h->stream));
    *used = o;
    return DBEC_OK;
}

// Every member's scalar block at create time: s = 1, G and D of the parameters, no ramp.
static int init_scalars(dbec_handle h) {
    std::vector<double> v((size_t)h->nb * SC_COUNT, 0.0);
    for (int b = 0; b < h->nb; ++b) {
        double* sc = v.data() + (size_t)b * SC_COUNT;
        sc[SC_S] = 1.0; sc[SC_S2] = 1.0; sc[SC_G] = h->p.G; sc[SC_D] = h->p.D;
    }
    CU(h, cudaMemcpyAsync(h->scal, v.data(), v.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    return DBEC_OK;
}

// Columns [first, first + count) of every member's scalar block <- vals[member][count] (HOST).
static int write_member_scalars(dbec_handle h, int first, int count, const double* vals) {
    CU(h, cudaMemcpy2DAsync(h->scal + first, SC_COUNT * sizeof(double), vals, count * sizeof(double), count * sizeof(double),
                            h->nb, cudaMemcpyHostToDevice, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    return DBEC_OK;
}

// Kernel slots of one step (dbec_step_profile / dbec_kernel_name).
enum { KS_DENS_FFTX = 0, KS_FFT_Y_FWD, KS_FFT_LAST_FMI, KS_FFT_Y_INV, KS_IFFTX_NONLIN, KS_CN_X, KS_CN_Y, KS_CN_Z, KS_SMALL_STEP };
static const char* const kernel_names[DBEC_MAX_KERNELS] = {
    "density+fft_x", "fft_y<fwd>", "fft_last<fwd*Vdd*inv>", "fft_y<inv>",
    "ifft_x+calcnu+cn_x", "cn_x", "cn_y", "cn_z", "sscn_step<cluster>"};
static_assert(DBEC_MAX_KERNELS == DBEC_KERNEL_SLOTS, "include/dbec.h and dbec_internal.hpp disagree on the slot count");

#define KLAUNCH(h, slot, x)                                                                      \
    do {                                                                                         \
        if ((h)->prof_on) cudaEventRecord((h)->prof_ev[2 * (h)->prof_n], (h)->stream);           \
        int rc_ = (x);                                                                           \
        if (rc_) return cuda_fail(h, (cudaError_t)rc_);                                          \
        if ((h)->prof_on) {                                                                      \
            cudaEventRecord((h)->prof_ev[2 * (h)->prof_n + 1], (h)->stream);                     \
            (h)->prof_slot[(h)->prof_n++] = (slot);                                              \
        }                                                                                        \
    } while (0)

// rev: walk the tiles of a plane-ordered pass last to first, so that it starts on the planes the
// previous pass has just left (dirty) in the 126 MB L2.
static int launch_fft_pass(dbec_handle h, int axis, int mode, int rev = 0) {
    h->rev_next = rev && h->use_rev;
    if (h->gen[axis]) return dbec_launch_gen_fft(h, axis, mode);
    return dbec_tma_supported(h, axis) ? dbec_launch_fft_tma(h, axis, mode, 0, h->nplanes) : dbec_launch_fft_strided(h, axis, mode);
}
static int launch_cn_pass(dbec_handle h, int axis, int with_norm, int rev = 0) {
    h->rev_next = rev && h->use_rev;
    if (h->gen[axis]) return dbec_launch_gen_cn(h, axis, with_norm);
    if (axis > 0 && dbec_tma_supported(h, axis)) {
        // a batch: the tiles of one CTA of the persistent sweep span several members, so calcnorm takes a
        // pass of its own (the fields of a batch are small: it runs out of L2)
        if (with_norm && h->nb > 1) {
            int rc = dbec_launch_cn_tma(h, axis, 0, 0, h->nplanes);
            return rc ? rc : dbec_launch_norm_only(h);
        }
        return dbec_launch_cn_tma(h, axis, with_norm, 0, h->nplanes);
    }
    return dbec_launch_cn(h, axis, with_norm);
}

// calcpsidd2 up to the x-inverse: density -> half spectrum -> x V_dd -> back along z, y.
// advance: 1 inside a step (the density pass also moves the NSTP ramp on, reading S26).
static int enqueue_dipolar_spectrum(dbec_handle h, int advance) {
    h->rev_next = 0;
    if (h->gen[0]) KLAUNCH(h, KS_DENS_FFTX, dbec_launch_gen_density_fftx(h, advance));
    else if (dbec_xline_supported(h)) KLAUNCH(h, KS_DENS_FFTX, dbec_launch_xline_density(h, 0, h->nplanes, advance));
    else KLAUNCH(h, KS_DENS_FFTX, dbec_launch_density_fftx(h, advance));
    if (h->p.ndim == 3) {
        KLAUNCH(h, KS_FFT_Y_FWD, launch_fft_pass(h, 1, 0, 1));      // density pass went up in z: come back down
        KLAUNCH(h, KS_FFT_LAST_FMI, launch_fft_pass(h, 2, 2));
        KLAUNCH(h, KS_FFT_Y_INV, launch_fft_pass(h, 1, 1));
    } else {
        KLAUNCH(h, KS_FFT_LAST_FMI, launch_fft_pass(h, 1, 2));
    }
    return DBEC_OK;
}

// One SSCN step as a sequence of launches (reading S10).
static int enqueue_step(dbec_handle h) {
    const bool imag = h->p.time_mode == 0;
    const int last_axis = h->p.ndim == 3 ? 2 : 1;
    int rc = enqueue_dipolar_spectrum(h, 1);
    if (rc) return rc;
    h->rev_next = h->use_rev;                                       // inverse y pass went up: come back down
    if (h->gen[0]) KLAUNCH(h, KS_IFFTX_NONLIN, dbec_launch_gen_nonlinear(h));
    else if (dbec_xwarp_supported(h)) KLAUNCH(h, KS_IFFTX_NONLIN, dbec_launch_xwarp_nonlin(h));
    else if (h->fuse_cnx && dbec_xline_supported(h)) KLAUNCH(h, KS_IFFTX_NONLIN, dbec_launch_xline_nonlin(h, 0, h->nplanes));
    else KLAUNCH(h, KS_IFFTX_NONLIN, dbec_launch_nonlinear(h, h->fuse_cnx));
    if (!h->fuse_cnx) KLAUNCH(h, KS_CN_X, launch_cn_pass(h, 0, 0));
    for (int ax = 1; ax <= last_axis; ++ax)
        KLAUNCH(h, ax == 1 ? KS_CN_Y : KS_CN_Z, launch_cn_pass(h, ax, imag && ax == last_axis));
    return DBEC_OK;
}

extern "C" {

int dbec_version(void) { return DBEC_VERSION; }

const char* dbec_strerror(int code) {
    switch (code) {
        case DBEC_OK: return "ok";
        case DBEC_EINVAL: return "invalid argument";
        case DBEC_ESIZE: return "unsupported grid length (4..1024 with prime factors 2, 3, 5, 7; NX and NY*NZ even)";
        case DBEC_EWORKSPACE: return "workspace missing, misaligned or too small";
        case DBEC_ECUDA: return "CUDA error (see dbec_last_cuda_error)";
        case DBEC_ENODEVICE: return "no sm_100 CUDA device";
        case DBEC_ENOALLOC_SIZE: return "dbec_norm_noalloc: more points than DBEC_NOALLOC_MAX_POINTS (2^27)";
        default: return "unknown error";
    }
}

int dbec_workspace_bytes_batch(const dbec_params* p, int nbatch, size_t* bytes) {
    if (!bytes || nbatch < 1 || nbatch > DBEC_MAX_BATCH) return DBEC_EINVAL;
    int rc = check_params(p);
    if (rc) return rc;
    Layout L;
    make_layout(p, nbatch, &L);
    *bytes = L.total;
    return DBEC_OK;
}

int dbec_workspace_bytes(const dbec_params* p, size_t* bytes) { return dbec_workspace_bytes_batch(p, 1, bytes); }

int dbec_create(const dbec_params* p, void* dev_workspace, size_t bytes, void* cuda_stream, dbec_handle* out) {
    return dbec_create_batch(p, 1, dev_workspace, bytes, cuda_stream, out);
}

int dbec_create_batch(const dbec_params* p, int nbatch, void* dev_workspace, size_t bytes, void* cuda_stream,
                      dbec_handle* out) {
    if (!out) return DBEC_EINVAL;
    *out = nullptr;
    if (nbatch < 1 || nbatch > DBEC_MAX_BATCH) return DBEC_EINVAL;
    int rc = check_params(p);
    if (rc) return rc;
    Layout L;
    make_layout(p, nbatch, &L);
    if (!dev_workspace || ((uintptr_t)dev_workspace & 255) || bytes < L.total) return DBEC_EWORKSPACE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return DBEC_ENODEVICE;
    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return DBEC_ENODEVICE;
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (major != 10) return DBEC_ENODEVICE;          // sm_100a code only, no fallback

    dbec_handle h = new (std::nothrow) dbec_handle_s();
    if (!h) return DBEC_EINVAL;
    cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev);
    h->p = *p;
    h->stream = (cudaStream_t)cuda_stream;
    h->nx = p->nx; h->ny = p->ny; h->nz = p->nz;
    h->nxhp = ((p->nx / 2 + 1) + DBEC_SPEC_COLS - 1) / DBEC_SPEC_COLS * DBEC_SPEC_COLS;
    h->P = (long long)p->nx * p->ny * p->nz;
    h->SP = (long long)p->nz * p->ny * h->nxhp;
    h->dV = p->ndim == 3 ? p->dx * p->dy * p->dz : p->dx * p->dy;
    h->nyf = p->ny / 2 + 1;
    h->nzf = p->nz / 2 + 1;
    h->nb = nbatch;
    h->nplanes = p->nz * nbatch;
    char* w = (char*)dev_workspace;
    h->psi = (cd*)(w + L.psi);
    h->spec = (cd*)(w + L.spec);
    h->vdd = (double*)(w + L.vdd);
    h->phi = (double*)(w + L.phi);
    h->scal = (double*)(w + L.scal);
    h->partial = (double*)(w + L.partial);
    h->ticket = (unsigned int*)(w + L.ticket);
    h->obs_dev = (double*)(w + L.obs);
    h->npartial = (int)L.npartial;
    // the only four switches (all exercised by tests/test_gpu_parity.py): the CUDA graph of a step, the x sweep
    // fused into the nonlinear kernel, the one-launch step of small grids (DBEC_CLUSTER: CTAs per cluster; 0 = off) and
    // the pacing of the streaming passes (DBEC_PACE, below)
    const char* fe = getenv("DBEC_FUSE_CNX");
    h->fuse_cnx = fe ? atoi(fe) : 1;
    const char* ge = getenv("DBEC_GRAPH");
    h->use_graph = ge ? atoi(ge) : 1;
    h->use_rev = 1; h->use_pdl = 1; h->use_tma = 1;
    h->zpair_min_stride = 2LL << 20;
    {   // Pacing of the streaming passes (tma_pipe.cuh: pace_wait).  The schedule interval is set by the THEORETICAL
        // DRAM bandwidth (B200: 2 x 3996 MHz x 7680 bit = 7672 GB/s), which no pass reaches: every CTA is then
        // "late", publishes its lag, and the loaders issue tile i when the slowest CTA of the launch has issued its
        // own — lockstep at whatever rate the memory delivers, with no tuned constant.  Scanned on B200: 5600 ...
        // 6600 GB/s has a sharp optimum at 6200 without the shared lag; with it, anything from 6800 up gives the
        // same step time (C5 2.25 -> 2.00 ms, C4 491 -> 478 us).  DBEC_PACE (GB/s; 0 = off) is the tests' switch.
        int khz = 0, bits = 0, l2 = 0;
        cudaDeviceGetAttribute(&khz, cudaDevAttrMemoryClockRate, dev);
        cudaDeviceGetAttribute(&bits, cudaDevAttrGlobalMemoryBusWidth, dev);
        cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev);
        h->l2_bytes = l2;
        h->pace_gbs = 2.0 * (double)khz * 1e3 * (double)bits / 8.0 / 1e9;
        h->pace_head_speed = 0.5;
        const char* pe = getenv("DBEC_PACE");
        if (pe) h->pace_gbs = atof(pe);
    }
    // the legacy default stream cannot be captured: plain launches there
    if (h->stream == nullptr || h->stream == cudaStreamLegacy) h->use_graph = 0;

    // a failed create has no handle to ask: its CUDA error is kept per thread (dbec_last_cuda_error(NULL))
#define FAIL(code) do { create_cuda_error = h->last_cuda ? h->last_cuda : (int)cudaGetLastError(); delete h; return (code); } while (0)
#define TRY(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { h->last_cuda = (int)e_; FAIL(DBEC_ECUDA); } } while (0)
    create_cuda_error = 0;
    TRY(cudaMemsetAsync(h->psi, 0, sizeof(cd) * h->P * h->nb, h->stream));
    TRY(cudaMemsetAsync(h->ticket, 0, 256, h->stream));
    TRY(cudaMemsetAsync(h->spec, 0, sizeof(cd) * h->SP * h->nb, h->stream));
    char* t = w + L.tables;
    const double om[3] = {p->nu, p->lambda, p->kappa};
    const double dd[3] = {p->dx, p->dy, p->ndim == 3 ? p->dz : 1.0};
    const int nn[3] = {p->nx, p->ny, p->nz};
    for (int ax = 0; ax < 3; ++ax) {
        h->gen[ax] = nn[ax] > 1 && !len_pow2_fast(nn[ax]);
        h->gnfac[ax] = h->gen[ax] ? dbec_gen_factor(nn[ax], h->gfac[ax]) : 0;
    }
    if (h->gen[0]) h->fuse_cnx = 0;               // the run-time-length nonlinear kernel carries no x sweep
    for (int ax = 0; ax < 3; ++ax) {
        size_t used = 0;
        rc = upload_axis(h, ax, nn[ax], dd[ax], (p->ndim == 2 && ax == 2) ? 0.0 : om[ax], t, &used);
        if (rc) FAIL(rc);
        t += used;
    }
    {
        const char* ce = getenv("DBEC_CLUSTER");
        int req = ce ? atoi(ce) : -1;
        if (req > 0 && req != 1 && req != 2 && req != 4 && req != 8 && req != 16) req = -1;
        h->use_cluster = dbec_small_choose(h, req);
        h->use_small = h->use_cluster > 0;
        // the automatic choice takes the compiled power-of-two variant where there is one (DBEC_SMALL_P2=0: never;
        // DBEC_SMALL_P2_CS=1, 4, 8, 16: only with that many CTAs per cluster)
        const char* p2 = getenv("DBEC_SMALL_P2");
        const char* p2cs = getenv("DBEC_SMALL_P2_CS");
        h->use_small_p2 = 0;
        if (req < 0 && !(p2 && atoi(p2) == 0)) {
            const int cs = dbec_small_p2_choose(h, p2cs ? atoi(p2cs) : -1);
            if (cs > 0) { h->use_small_p2 = 1; h->use_small = 1; h->use_cluster = cs; }
        }
    }
    if (h->use_tma) TRY((cudaError_t)dbec_make_tensor_maps(h));
    if (init_scalars(h)) FAIL(DBEC_ECUDA);
    TRY((cudaError_t)dbec_launch_build_vdd(h));
    TRY(cudaStreamSynchronize(h->stream));
#undef TRY
#undef FAIL
    *out = h;
    return DBEC_OK;
}

int dbec_destroy(dbec_handle h) {
    if (!h) return DBEC_EINVAL;
    cudaStreamSynchronize(h->stream);
    if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
    delete h;
    return DBEC_OK;
}

int dbec_last_cuda_error(dbec_handle h) { return h ? h->last_cuda : create_cuda_error; }

const char* dbec_build_id(void) {
#ifndef DBEC_BUILD_ID_STR
#define DBEC_BUILD_ID_STR "unknown"
#endif
    return "DBEC_BUILD_ID=" DBEC_BUILD_ID_STR;
}

int dbec_set_psi(dbec_handle h, const void* psi, int on_device) {
    if (!h || !psi) return DBEC_EINVAL;
    CU(h, cudaMemcpyAsync(h->psi, psi, sizeof(cd) * h->P * h->nb, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice,
                          h->stream));
    // a fresh field carries no deferred norm factor
    LAUNCH(h, dbec_launch_reset_scale(h));
    if (!on_device) CU(h, cudaStreamSynchronize(h->stream));
    return DBEC_OK;
}

int dbec_get_psi(dbec_handle h, void* psi, int on_device) {
    if (!h || !psi) return DBEC_EINVAL;
    if (h->p.time_mode == 0) LAUNCH(h, dbec_launch_apply_scale(h));     // s is 1 for ever in real time
    CU(h, cudaMemcpyAsync(psi, h->psi, sizeof(cd) * h->P * h->nb, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                          h->stream));
    if (!on_device) CU(h, cudaStreamSynchronize(h->stream));
    return DBEC_OK;
}

int dbec_set_psi_async(dbec_handle h, const void* psi) {
    if (!h || !psi) return DBEC_EINVAL;
    CU(h, cudaMemcpyAsync(h->psi, psi, sizeof(cd) * h->P * h->nb, cudaMemcpyHostToDevice, h->stream));
    LAUNCH(h, dbec_launch_reset_scale(h));             // a fresh field carries no deferred norm factor
    return DBEC_OK;
}

int dbec_get_psi_async(dbec_handle h, void* psi) {
    if (!h || !psi) return DBEC_EINVAL;
    if (h->p.time_mode == 0) LAUNCH(h, dbec_launch_apply_scale(h));
    CU(h, cudaMemcpyAsync(psi, h->psi, sizeof(cd) * h->P * h->nb, cudaMemcpyDeviceToHost, h->stream));
    return DBEC_OK;
}

int dbec_synchronize(dbec_handle h) {
    if (!h) return DBEC_EINVAL;
    CU(h, cudaStreamSynchronize(h->stream));
    return DBEC_OK;
}

// Columns SC_G .. SC_RN of every member: the current (G, D), then a ramp G0, D0, G1, D1, k = 0, n.
static int write_couplings(dbec_handle h, const double* G, int gs, const double* D, int ds, int nstp, const double* G0,
                           const double* D0) {
    const int cols = SC_RN - SC_G + 1;
    std::vector<double> v((size_t)h->nb * cols);
    for (int b = 0; b < h->nb; ++b) {
        double* r = v.data() + (size_t)b * cols;
        const double g1 = G[b * gs], d1 = D[b * ds];
        const double g0 = nstp > 0 ? G0[0] : g1, d0 = nstp > 0 ? D0[0] : d1;
        r[SC_G - SC_G] = g0; r[SC_D - SC_G] = d0;
        r[SC_G0 - SC_G] = g0; r[SC_D0 - SC_G] = d0; r[SC_G1 - SC_G] = g1; r[SC_D1 - SC_G] = d1;
        r[SC_RK - SC_G] = 0.0; r[SC_RN - SC_G] = (double)nstp;
    }
    return write_member_scalars(h, SC_G, cols, v.data());
}

int dbec_set_coupling(dbec_handle h, double G, double D) {
    if (!h) return DBEC_EINVAL;
    h->p.G = G; h->p.D = D;
    return write_couplings(h, &G, 0, &D, 0, 0, nullptr, nullptr);
}

int dbec_set_coupling_batch(dbec_handle h, const double* G, const double* D) {
    if (!h || !G || !D) return DBEC_EINVAL;
    return write_couplings(h, G, 1, D, 1, 0, nullptr, nullptr);
}

int dbec_set_ramp(dbec_handle h, int nstp, double G0, double D0, double G1, double D1) {
    if (!h || nstp < 0) return DBEC_EINVAL;
    h->p.G = G1; h->p.D = D1;
    return write_couplings(h, &G1, 0, &D1, 0, nstp, &G0, &D0);
}

int dbec_batch_size(dbec_handle h, int* nbatch) {
    if (!h || !nbatch) return DBEC_EINVAL;
    *nbatch = h->nb;
    return DBEC_OK;
}

int dbec_step(dbec_handle h, int nsteps) {
    if (!h || nsteps < 0) return DBEC_EINVAL;
    if (h->use_small) {
        // a small grid: one launch runs all nsteps steps inside one thread-block cluster (kernels_small.cu)
        if (nsteps > 0) LAUNCH(h, dbec_launch_small_step(h, nsteps));
        return DBEC_OK;
    }
    if (!h->use_graph) {
        for (int i = 0; i < nsteps; ++i) { int rc = enqueue_step(h); if (rc) return rc; }
        return DBEC_OK;
    }
    if (!h->graph_exec) {
        // warm every kernel once outside capture is not needed: launches inside a capture are recorded,
        // not executed; function attributes (dynamic shared memory) are set by the launchers up front.
        cudaGraph_t g = nullptr;
        const long long before = h->launches;
        CU(h, cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
        int rc = enqueue_step(h);
        cudaError_t e = cudaStreamEndCapture(h->stream, &g);
        h->launches_per_step = (int)(h->launches - before);
        h->launches = before;
        if (rc) { if (g) cudaGraphDestroy(g); return rc; }
        if (e != cudaSuccess) return cuda_fail(h, e);
        e = cudaGraphInstantiate(&h->graph_exec, g, 0);
        cudaGraphDestroy(g);
        if (e != cudaSuccess) return cuda_fail(h, e);
    }
    for (int i = 0; i < nsteps; ++i) {
        CU(h, cudaGraphLaunch(h->graph_exec, h->stream));
        h->launches += h->launches_per_step;
    }
    return DBEC_OK;
}

int dbec_phi_dd(dbec_handle h, void* phi_f64_dev) {
    if (!h || !phi_f64_dev) return DBEC_EINVAL;
    { int rc = enqueue_dipolar_spectrum(h, 0); if (rc) return rc; }
    LAUNCH(h, h->gen[0] ? dbec_launch_gen_phi_out(h, (double*)phi_f64_dev) : dbec_launch_phi_out(h, (double*)phi_f64_dev));
    return DBEC_OK;
}

int dbec_cn_sweep(dbec_handle h, int axis) {
    if (!h || axis < 0 || axis > 2 || (h->p.ndim == 2 && axis == 2)) return DBEC_EINVAL;
    LAUNCH(h, launch_cn_pass(h, axis, 0));
    return DBEC_OK;
}

int dbec_nonlinear(dbec_handle h) {
    if (!h) return DBEC_EINVAL;
    // the nonlinear kernel multiplies by the deferred norm factor s but leaves it in place (inside a step the
    // last sweep rewrites it): bring the stored field to s = 1 first, or every later consumer applies s again
    LAUNCH(h, dbec_launch_apply_scale(h));
    { int rc = enqueue_dipolar_spectrum(h, 0); if (rc) return rc; }
    LAUNCH(h, h->gen[0] ? dbec_launch_gen_nonlinear(h) : dbec_launch_nonlinear(h, 0));
    return DBEC_OK;
}

int dbec_normalize(dbec_handle h) {
    if (!h) return DBEC_EINVAL;
    LAUNCH(h, dbec_launch_normalize(h));
    // real time never rewrites the factor (no calcnorm inside its step) and dbec_get_psi does not apply it:
    // apply it now, so that s is 1 again and the field stays normalised instead of being rescaled every step
    if (h->p.time_mode == 1) LAUNCH(h, dbec_launch_apply_scale(h));
    return DBEC_OK;
}

int dbec_observables_batch(dbec_handle h, dbec_obs* out) {
    if (!h || !out) return DBEC_EINVAL;
    { int rc = enqueue_dipolar_spectrum(h, 0); if (rc) return rc; }
    LAUNCH(h, h->gen[0] ? dbec_launch_gen_phi_out(h, h->phi) : dbec_launch_phi_out(h, h->phi));
    LAUNCH(h, dbec_launch_observables(h));
    std::vector<double> v((size_t)h->nb * 16);
    CU(h, cudaMemcpyAsync(v.data(), h->obs_dev, v.size() * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    for (int b = 0; b < h->nb; ++b) {
        const double* r = v.data() + (size_t)b * 16;
        dbec_obs& o = out[b];
        o.norm = r[0]; o.mu = r[1]; o.energy = r[2];
        o.rms_x = r[3]; o.rms_y = r[4]; o.rms_z = r[5]; o.rms_r = r[6];
        o.density0 = r[7]; o.density_max = r[8];
    }
    return DBEC_OK;
}

int dbec_observables(dbec_handle h, dbec_obs* out) {
    if (!h || !out || h->nb != 1) return DBEC_EINVAL;      // a batch has one record per member: dbec_observables_batch
    return dbec_observables_batch(h, out);
}

// Integrated densities (reading S27).  The result is produced on the device; out may be HOST or DEVICE.
static int density_out(dbec_handle h, const double* dev, size_t count, void* out, int on_device) {
    CU(h, cudaMemcpyAsync(out, dev, count * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    if (!on_device) CU(h, cudaStreamSynchronize(h->stream));
    return DBEC_OK;
}

int dbec_density_1d(dbec_handle h, int member, int axis, double* out, int on_device) {
    if (!h || !out || member < 0 || member >= h->nb || axis < 0 || axis >= h->p.ndim) return DBEC_EINVAL;
    // h->phi (P doubles per member, scratch outside dbec_observables) holds the intermediate 2-D density and the result
    const int n[3] = {h->nx, h->ny, h->nz};
    double* scratch = h->phi;
    double* res = h->phi + (h->P - n[axis]);              // the tail of the first member's block: never overlaps a 2-D density
    LAUNCH(h, dbec_launch_density_1d(h, member, axis, res, scratch));
    return density_out(h, res, (size_t)n[axis], out, on_device);
}

int dbec_density_2d(dbec_handle h, int member, int axis_integrated, double* out, int on_device) {
    if (!h || !out || member < 0 || member >= h->nb || h->p.ndim != 3 || axis_integrated < 0 || axis_integrated > 2)
        return DBEC_EINVAL;
    const size_t count = (size_t)h->P / (size_t)(axis_integrated == 0 ? h->nx : axis_integrated == 1 ? h->ny : h->nz);
    LAUNCH(h, dbec_launch_density_2d(h, member, axis_integrated, h->phi));
    return density_out(h, h->phi, count, out, on_device);
}

// nsteps steps with plain launches and a CUDA event pair around every kernel.  ms_per_slot receives
// DBEC_MAX_KERNELS doubles: total milliseconds spent in each kernel slot over the nsteps steps;
// launches_per_slot the launch counts.  Synchronises the stream.
int dbec_step_profile(dbec_handle h, int nsteps, double* ms_per_slot, long long* launches_per_slot) {
    if (!h || nsteps < 0 || !ms_per_slot || !launches_per_slot) return DBEC_EINVAL;
    for (int i = 0; i < DBEC_MAX_KERNELS; ++i) { ms_per_slot[i] = 0.0; launches_per_slot[i] = 0; }
    for (int i = 0; i < 2 * DBEC_MAX_KERNELS; ++i) CU(h, cudaEventCreate(&h->prof_ev[i]));
    int rc = DBEC_OK;
    for (int s = 0; s < nsteps && rc == DBEC_OK; ++s) {
        h->prof_on = 1; h->prof_n = 0;
        if (h->use_small) {
            rc = [&]() -> int { KLAUNCH(h, KS_SMALL_STEP, dbec_launch_small_step(h, 1)); return DBEC_OK; }();
        } else {
            rc = enqueue_step(h);
        }
        h->prof_on = 0;
        if (rc) break;
        if (cudaStreamSynchronize(h->stream) != cudaSuccess) { rc = DBEC_ECUDA; break; }
        for (int k = 0; k < h->prof_n; ++k) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, h->prof_ev[2 * k], h->prof_ev[2 * k + 1]);
            ms_per_slot[h->prof_slot[k]] += ms;
            launches_per_slot[h->prof_slot[k]] += 1;
        }
    }
    for (int i = 0; i < 2 * DBEC_MAX_KERNELS; ++i) cudaEventDestroy(h->prof_ev[i]);
    return rc;
}

const char* dbec_kernel_name(int slot) {
    return (slot >= 0 && slot < DBEC_MAX_KERNELS) ? kernel_names[slot] : "";
}

// Which __global__ function serves a pass of dbec_step on this handle (lines of 128..512 points go to the
// persistent TMA / bulk-copy kernels, shorter ones to the one-tile-per-block kernels; a small grid's whole step
// is one launch of k_small_step).
const char* dbec_pass_kernel(dbec_handle h, int slot) {
    if (!h || slot < 0 || slot >= DBEC_MAX_KERNELS) return "";
    const int last_axis = h->p.ndim == 3 ? 2 : 1;
    if (h->use_small) return slot == KS_SMALL_STEP ? (h->use_small_p2 ? "k_small_p2" : "k_small_step") : "";      // dbec_step launches nothing else
    switch (slot) {
        case KS_DENS_FFTX: return h->gen[0] ? "k_gen_density_fftx" : dbec_xline_supported(h) ? "k_xline_density" : "k_density_fftx";
        case KS_FFT_Y_FWD: case KS_FFT_Y_INV:
            return h->p.ndim == 3 ? (h->gen[1] ? "k_gen_fft_strided" : dbec_tma_supported(h, 1) ? "k_fft_tma" : "k_fft_strided") : "";
        case KS_FFT_LAST_FMI:
            return h->gen[last_axis] ? "k_gen_fft_strided" : dbec_tma_supported(h, last_axis) ? "k_fft_tma" : "k_fft_strided";
        case KS_IFFTX_NONLIN: return h->gen[0] ? "k_gen_ifftx_nonlin" : dbec_xwarp_supported(h) ? "k_xwarp_nonlin"
                                     : (h->fuse_cnx && dbec_xline_supported(h)) ? "k_xline_nonlin" : "k_ifftx_nonlin";
        case KS_CN_X: return h->fuse_cnx ? "" : h->gen[0] ? "k_gen_cn" : "k_cn_x";
        case KS_CN_Y: return h->gen[1] ? "k_gen_cn" : dbec_tma_supported(h, 1) ? "k_cn_tma" : "k_cn_strided";
        case KS_CN_Z: return h->p.ndim == 3 ? (h->gen[2] ? "k_gen_cn" : dbec_tma_supported(h, 2) ? "k_cn_tma" : "k_cn_strided") : "";
    }
    return "";
}

int dbec_launch_count(dbec_handle h, long long* launches) {
    if (!h || !launches) return DBEC_EINVAL;
    *launches = h->launches;
    return DBEC_OK;
}

}  // extern "C"
