"""Thin Python binding of libdbec.so (include/dbec.h): argument marshalling only.

torch is used for device memory (the workspace the caller owns) and the CUDA stream; every step of
the path runs in the library's sm_100a kernels.  There is no CPU fallback: importing works without a
GPU (so that the symbols can be checked), creating a simulation does not.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdbec.so")

DBEC_OK, DBEC_EINVAL, DBEC_ESIZE, DBEC_EWORKSPACE, DBEC_ECUDA, DBEC_ENODEVICE = 0, -1, -2, -3, -4, -5

EXPORTS = ["dbec_workspace_bytes", "dbec_create", "dbec_set_psi", "dbec_get_psi", "dbec_set_coupling",
           "dbec_step", "dbec_observables", "dbec_destroy", "dbec_strerror", "dbec_last_cuda_error",
           "dbec_phi_dd", "dbec_cn_sweep", "dbec_nonlinear", "dbec_normalize", "dbec_launch_count",
           "dbec_version", "dbec_step_profile", "dbec_kernel_name", "dbec_pass_kernel", "dbec_build_id",
           "dbec_set_ramp", "dbec_workspace_bytes_batch", "dbec_create_batch", "dbec_batch_size",
           "dbec_set_coupling_batch", "dbec_observables_batch", "dbec_density_1d", "dbec_density_2d",
           "dbec_norm_noalloc", "dbec_noalloc_last_cuda_error", "dbec_set_psi_async", "dbec_get_psi_async",
           "dbec_synchronize"]
KERNEL_SLOTS = 9


class DbecParams(C.Structure):
    _fields_ = [("ndim", C.c_int32), ("plane", C.c_int32),
                ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("dt", C.c_double),
                ("nu", C.c_double), ("lam", C.c_double), ("kappa", C.c_double),
                ("G", C.c_double), ("D", C.c_double),
                ("d_perp", C.c_double), ("cutoff", C.c_double),
                ("time_mode", C.c_int32)]


class DbecObs(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("norm", "mu", "energy", "rms_x", "rms_y", "rms_z", "rms_r", "density0", "density_max")]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class DbecError(RuntimeError):
    def __init__(self, code, what, cuda=0):
        self.code = code
        self.cuda = cuda
        msg = lib().dbec_strerror(code).decode()
        super().__init__(f"{what}: {msg} (code {code}" + (f", CUDA error {cuda})" if cuda else ")"))


_lib = None


def lib():
    """Load libdbec.so (building it in-tree with nvcc if it is missing or was built from other sources:
    build() compares the source hash inside the library with the tree and is a no-op when they agree)."""
    global _lib
    if _lib is None:
        _build.build()
        L = C.CDLL(LIB_PATH)
        pp, vp = C.POINTER(DbecParams), C.c_void_p
        L.dbec_workspace_bytes.argtypes = [pp, C.POINTER(C.c_size_t)]
        L.dbec_create.argtypes = [pp, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.dbec_set_psi.argtypes = [vp, vp, C.c_int]
        L.dbec_get_psi.argtypes = [vp, vp, C.c_int]
        L.dbec_set_coupling.argtypes = [vp, C.c_double, C.c_double]
        L.dbec_step.argtypes = [vp, C.c_int]
        L.dbec_observables.argtypes = [vp, C.POINTER(DbecObs)]
        L.dbec_destroy.argtypes = [vp]
        L.dbec_strerror.argtypes = [C.c_int]
        L.dbec_strerror.restype = C.c_char_p
        L.dbec_last_cuda_error.argtypes = [vp]
        L.dbec_phi_dd.argtypes = [vp, vp]
        L.dbec_cn_sweep.argtypes = [vp, C.c_int]
        L.dbec_nonlinear.argtypes = [vp]
        L.dbec_normalize.argtypes = [vp]
        L.dbec_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.dbec_version.argtypes = []
        L.dbec_step_profile.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.dbec_kernel_name.argtypes = [C.c_int]
        L.dbec_kernel_name.restype = C.c_char_p
        L.dbec_pass_kernel.argtypes = [vp, C.c_int]
        L.dbec_pass_kernel.restype = C.c_char_p
        dp = C.POINTER(C.c_double)
        L.dbec_set_ramp.argtypes = [vp, C.c_int] + [C.c_double] * 4
        L.dbec_workspace_bytes_batch.argtypes = [pp, C.c_int, C.POINTER(C.c_size_t)]
        L.dbec_create_batch.argtypes = [pp, C.c_int, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.dbec_batch_size.argtypes = [vp, C.POINTER(C.c_int)]
        L.dbec_set_coupling_batch.argtypes = [vp, dp, dp]
        L.dbec_observables_batch.argtypes = [vp, C.POINTER(DbecObs)]
        L.dbec_density_1d.argtypes = [vp, C.c_int, C.c_int, vp, C.c_int]
        L.dbec_density_2d.argtypes = [vp, C.c_int, C.c_int, vp, C.c_int]
        L.dbec_set_psi_async.argtypes = [vp, vp]
        L.dbec_get_psi_async.argtypes = [vp, vp]
        L.dbec_synchronize.argtypes = [vp]
        L.dbec_build_id.argtypes = []
        L.dbec_build_id.restype = C.c_char_p
        L.dbec_norm_noalloc.argtypes = [vp, C.c_longlong, C.c_double, vp, vp]
        L.dbec_noalloc_last_cuda_error.argtypes = []
        _lib = L
    return _lib


def params(ndim, nx, ny, nz, dx, dy, dz, dt, nu, lam, kappa, G, D, time_mode,
           d_perp=1.0, cutoff=0.0, plane=0) -> DbecParams:
    return DbecParams(ndim, plane, nx, ny, nz, dx, dy, dz, dt, nu, lam, kappa, G, D, d_perp, cutoff, time_mode)


def params_of(w, G=None, D=None) -> DbecParams:
    """DbecParams from an object with the attribute names of inputs.Workload (duck-typed)."""
    return params(w.ndim, w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.dt, w.nu, w.lam, w.kappa,
                  w.G if G is None else G, w.D if D is None else D, w.time_mode,
                  d_perp=w.d_perp, cutoff=w.cutoff, plane=getattr(w, "plane", 0))


def workspace_bytes(p: DbecParams, nbatch: int = 1) -> int:
    n = C.c_size_t(0)
    rc = lib().dbec_workspace_bytes_batch(C.byref(p), int(nbatch), C.byref(n))
    if rc:
        raise DbecError(rc, "dbec_workspace_bytes_batch")
    return int(n.value)


class Dbec:
    """One simulation (or a batch of `nbatch` independent ones with the same parameters) behind the C ABI."""

    def __init__(self, p: DbecParams, device="cuda:0", stream=None, nbatch: int = 1):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1601_04640_b200 needs a CUDA device (sm_100a); there is no CPU path")
        self._torch = torch
        self.p = p
        self.nbatch = int(nbatch)
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        # a stream of its own by default: the step is replayed as a CUDA graph, which the legacy default
        # stream cannot capture
        self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
        nbytes = workspace_bytes(p, self.nbatch)
        # caller-owned workspace; torch allocations are 512-byte aligned
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        assert self.workspace.data_ptr() % 256 == 0
        self._h = C.c_void_p()
        rc = lib().dbec_create_batch(C.byref(p), self.nbatch, C.c_void_p(self.workspace.data_ptr()), nbytes,
                                     C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if rc:
            raise DbecError(rc, "dbec_create_batch", lib().dbec_last_cuda_error(None))
        self.grid_shape = (p.nz, p.ny, p.nx) if p.ndim == 3 else (p.ny, p.nx)
        self.shape = self.grid_shape if self.nbatch == 1 else (self.nbatch,) + self.grid_shape
        self.npoints = p.nx * p.ny * p.nz * self.nbatch

    # -- helpers
    def _ck(self, rc, what):
        if rc:
            raise DbecError(rc, what, lib().dbec_last_cuda_error(self._h) if self._h else 0)

    def close(self):
        if getattr(self, "_h", None):
            lib().dbec_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ptr(self, a):
        """(pointer, on_device) of a numpy array or a torch tensor holding npoints complex128."""
        torch = self._torch
        if isinstance(a, np.ndarray):
            assert a.dtype == np.complex128 and a.flags.c_contiguous and a.size == self.npoints
            return a.ctypes.data, 0
        assert a.dtype == torch.complex128 and a.is_contiguous() and a.numel() == self.npoints
        return a.data_ptr(), 1 if a.is_cuda else 0

    # -- C entry points
    def set_psi(self, psi):
        if isinstance(psi, np.ndarray):
            psi = np.ascontiguousarray(psi, dtype=np.complex128)
        ptr, dev = self._ptr(psi)
        if dev:
            self.stream.wait_stream(self._torch.cuda.current_stream(self.device))
        self._ck(lib().dbec_set_psi(self._h, C.c_void_p(ptr), dev), "dbec_set_psi")

    def get_psi(self, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=np.complex128)
        ptr, dev = self._ptr(out)
        if dev:
            self.stream.wait_stream(self._torch.cuda.current_stream(self.device))
        self._ck(lib().dbec_get_psi(self._h, C.c_void_p(ptr), dev), "dbec_get_psi")
        if dev:
            self._torch.cuda.current_stream(self.device).wait_stream(self.stream)
        return out

    def set_psi_async(self, host):
        """dbec_set_psi_async: `host` a pinned CPU tensor / array of npoints complex128; returns at once."""
        ptr, dev = self._ptr(host)
        assert not dev, "set_psi_async takes a host buffer (device buffers: set_psi is asynchronous already)"
        self._ck(lib().dbec_set_psi_async(self._h, C.c_void_p(ptr)), "dbec_set_psi_async")

    def get_psi_async(self, host):
        """dbec_get_psi_async: the copy into `host` (pinned) is complete after wait()."""
        ptr, dev = self._ptr(host)
        assert not dev, "get_psi_async takes a host buffer"
        self._ck(lib().dbec_get_psi_async(self._h, C.c_void_p(ptr)), "dbec_get_psi_async")

    def wait(self):
        self._ck(lib().dbec_synchronize(self._h), "dbec_synchronize")

    def set_coupling(self, G, D):
        """Scalars: every member; sequences of nbatch values: per member."""
        if np.ndim(G) == 0 and np.ndim(D) == 0:
            self._ck(lib().dbec_set_coupling(self._h, float(G), float(D)), "dbec_set_coupling")
            return
        g = np.ascontiguousarray(np.broadcast_to(np.asarray(G, dtype=np.float64), (self.nbatch,)))
        d = np.ascontiguousarray(np.broadcast_to(np.asarray(D, dtype=np.float64), (self.nbatch,)))
        dp = C.POINTER(C.c_double)
        self._ck(lib().dbec_set_coupling_batch(self._h, g.ctypes.data_as(dp), d.ctypes.data_as(dp)), "dbec_set_coupling_batch")

    def set_ramp(self, nstp, G0, D0, G1, D1):
        self._ck(lib().dbec_set_ramp(self._h, int(nstp), float(G0), float(D0), float(G1), float(D1)), "dbec_set_ramp")

    def step(self, n=1):
        self._ck(lib().dbec_step(self._h, int(n)), "dbec_step")

    def observables(self):
        """One dict (plain handle) or a list of nbatch dicts (batch handle)."""
        if self.nbatch == 1:
            o = DbecObs()
            self._ck(lib().dbec_observables(self._h, C.byref(o)), "dbec_observables")
            return o.as_dict()
        arr = (DbecObs * self.nbatch)()
        self._ck(lib().dbec_observables_batch(self._h, arr), "dbec_observables_batch")
        return [o.as_dict() for o in arr]

    def density_1d(self, axis, member=0) -> np.ndarray:
        out = np.empty((self.p.nx, self.p.ny, self.p.nz)[axis], dtype=np.float64)
        self._ck(lib().dbec_density_1d(self._h, int(member), int(axis), C.c_void_p(out.ctypes.data), 0), "dbec_density_1d")
        return out

    def density_2d(self, axis_integrated, member=0) -> np.ndarray:
        shp = [self.p.nz, self.p.ny, self.p.nx]
        del shp[2 - axis_integrated]
        out = np.empty(shp, dtype=np.float64)
        self._ck(lib().dbec_density_2d(self._h, int(member), int(axis_integrated), C.c_void_p(out.ctypes.data), 0),
                 "dbec_density_2d")
        return out

    def phi_dd(self):
        out = self._torch.empty(self.shape, dtype=self._torch.float64, device=self.device)
        self.stream.wait_stream(self._torch.cuda.current_stream(self.device))
        self._ck(lib().dbec_phi_dd(self._h, C.c_void_p(out.data_ptr())), "dbec_phi_dd")
        self._torch.cuda.current_stream(self.device).wait_stream(self.stream)
        return out

    def cn_sweep(self, axis):
        self._ck(lib().dbec_cn_sweep(self._h, int(axis)), "dbec_cn_sweep")

    def nonlinear(self):
        self._ck(lib().dbec_nonlinear(self._h), "dbec_nonlinear")

    def normalize(self):
        self._ck(lib().dbec_normalize(self._h), "dbec_normalize")

    def launch_count(self) -> int:
        n = C.c_longlong(0)
        self._ck(lib().dbec_launch_count(self._h, C.byref(n)), "dbec_launch_count")
        return int(n.value)

    def step_profile(self, n=1) -> dict:
        """{kernel name: (total ms, launches)} over n steps, CUDA events around every launch."""
        ms = (C.c_double * KERNEL_SLOTS)()
        cnt = (C.c_longlong * KERNEL_SLOTS)()
        self._ck(lib().dbec_step_profile(self._h, int(n), ms, cnt), "dbec_step_profile")
        return {lib().dbec_kernel_name(i).decode(): (ms[i], cnt[i]) for i in range(KERNEL_SLOTS) if cnt[i]}

    def pass_kernels(self) -> dict:
        """{pass name: __global__ function serving it on this handle}."""
        out = {}
        for i in range(KERNEL_SLOTS):
            k = lib().dbec_pass_kernel(self._h, i).decode()
            if k:
                out[lib().dbec_kernel_name(i).decode()] = k
        return out

    def synchronize(self):
        self.stream.synchronize()


NOALLOC_MAX_POINTS = 1 << 27       # include/dbec.h: DBEC_NOALLOC_MAX_POINTS


def norm_noalloc(psi, dV: float, out=None, stream=None):
    """dbec_norm_noalloc: dV * sum |psi|^2 of a CUDA complex128 tensor, written into `out` (a one-element CUDA
    float64 tensor, made here if not given — the C call itself allocates nothing).  Asynchronous on `stream`
    (default: torch's current stream).  Calls that overlap on the GPU share one scratch array and race."""
    import torch
    assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous()
    if out is None:
        out = torch.empty(1, dtype=torch.float64, device=psi.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 1
    with torch.cuda.device(psi.device):
        st = stream if stream is not None else torch.cuda.current_stream(psi.device)
        rc = lib().dbec_norm_noalloc(psi.data_ptr(), psi.numel(), float(dV), out.data_ptr(), st.cuda_stream)
    if rc:
        raise DbecError(rc, "dbec_norm_noalloc", lib().dbec_noalloc_last_cuda_error())
    return out
