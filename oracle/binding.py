"""ctypes binding of oracle/dbec_oracle.cpp — TEST INFRASTRUCTURE, never on the product path.

`build()` compiles the C++ file with g++ (-O2 -fopenmp) into oracle/libdbec_oracle.so;
`Oracle` drives a state through the oracle's C ABI on host (numpy) memory.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dbec_oracle.cpp")
_LIB = os.path.join(_HERE, "libdbec_oracle.so")
_lib = None


class OracleParams(C.Structure):
    _fields_ = [("ndim", C.c_int32), ("plane", C.c_int32),
                ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("dt", C.c_double),
                ("nu", C.c_double), ("lam", C.c_double), ("kappa", C.c_double),
                ("G", C.c_double), ("D", C.c_double),
                ("d_perp", C.c_double), ("cutoff", C.c_double),
                ("time_mode", C.c_int32)]


class OracleObs(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("norm", "mu", "energy", "rms_x", "rms_y", "rms_z", "rms_r", "density0", "density_max")]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-fopenmp", "-std=c++17", "-shared", "-fPIC",
                               "-o", _LIB, _SRC])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        pp = C.POINTER(OracleParams)
        L.dbec_oracle_threads.restype = C.c_int
        L.dbec_oracle_create.argtypes = [pp, C.POINTER(C.c_void_p)]
        L.dbec_oracle_destroy.argtypes = [C.c_void_p]
        L.dbec_oracle_set_psi.argtypes = [C.c_void_p, dp]
        L.dbec_oracle_get_psi.argtypes = [C.c_void_p, dp]
        L.dbec_oracle_set_coupling.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.dbec_oracle_step.argtypes = [C.c_void_p, C.c_int]
        L.dbec_oracle_set_ramp.argtypes = [C.c_void_p, C.c_int] + [C.c_double] * 4
        L.dbec_oracle_get_coupling.argtypes = [C.c_void_p, dp, dp]
        L.dbec_oracle_density_1d.argtypes = [C.c_void_p, C.c_int, dp]
        L.dbec_oracle_density_2d.argtypes = [C.c_void_p, C.c_int, dp]
        L.dbec_oracle_observables.argtypes = [C.c_void_p, C.POINTER(OracleObs)]
        L.dbec_oracle_fft.argtypes = [dp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        L.dbec_oracle_erfcx.argtypes = [C.c_double]
        L.dbec_oracle_erfcx.restype = C.c_double
        L.dbec_oracle_vdd3d.argtypes = [C.c_double] * 4
        L.dbec_oracle_vdd3d.restype = C.c_double
        L.dbec_oracle_vdd2d.argtypes = [C.c_double] * 3
        L.dbec_oracle_vdd2d.restype = C.c_double
        L.dbec_oracle_vdd2d_xz.argtypes = [C.c_double] * 3
        L.dbec_oracle_vdd2d_xz.restype = C.c_double
        L.dbec_oracle_wavenumber.argtypes = [C.c_int, C.c_int, C.c_double]
        L.dbec_oracle_wavenumber.restype = C.c_double
        L.dbec_oracle_vdd_table.argtypes = [pp, dp]
        L.dbec_oracle_phi_dd.argtypes = [pp, dp, dp, C.c_int]
        L.dbec_oracle_nonlinear.argtypes = [pp, dp, dp]
        L.dbec_oracle_cn_sweep.argtypes = [pp, dp, C.c_int]
        L.dbec_oracle_cn_line.argtypes = [dp, C.c_int, C.c_double, C.c_double]
        L.dbec_oracle_normalize.argtypes = [pp, dp]
        L.dbec_oracle_norm.argtypes = [pp, dp]
        L.dbec_oracle_norm.restype = C.c_double
        _lib = L
    return _lib


def threads() -> int:
    return int(lib().dbec_oracle_threads())


def params(ndim, nx, ny, nz, dx, dy, dz, dt, nu, lam, kappa, G, D, time_mode,
           d_perp=1.0, cutoff=0.0, plane=0) -> OracleParams:
    return OracleParams(ndim, plane, nx, ny, nz, dx, dy, dz, dt, nu, lam, kappa, G, D,
                        d_perp, cutoff, time_mode)


def params_of(w, G=None, D=None) -> OracleParams:
    """OracleParams from any object with the Workload attribute names (duck-typed)."""
    return params(w.ndim, w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.dt, w.nu, w.lam, w.kappa,
                  w.G if G is None else G, w.D if D is None else D, w.time_mode,
                  d_perp=w.d_perp, cutoff=w.cutoff, plane=getattr(w, "plane", 0))


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128).copy()


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


class Oracle:
    """One simulation state in the oracle (host memory)."""

    def __init__(self, p: OracleParams):
        self.p = p
        self._h = C.c_void_p()
        _check(lib().dbec_oracle_create(C.byref(p), C.byref(self._h)), "create")
        self.shape = (p.nz, p.ny, p.nx) if p.ndim == 3 else (p.ny, p.nx)

    def close(self):
        if self._h:
            lib().dbec_oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_psi(self, psi):
        a = _c128(psi)
        assert a.size == self.p.nx * self.p.ny * self.p.nz
        _check(lib().dbec_oracle_set_psi(self._h, _dp(a)), "set_psi")

    def get_psi(self) -> np.ndarray:
        a = np.empty(self.shape, dtype=np.complex128)
        _check(lib().dbec_oracle_get_psi(self._h, _dp(a)), "get_psi")
        return a

    def set_coupling(self, G, D):
        _check(lib().dbec_oracle_set_coupling(self._h, G, D), "set_coupling")

    def step(self, n=1):
        _check(lib().dbec_oracle_step(self._h, int(n)), "step")

    def set_ramp(self, nstp, G0, D0, G1, D1):
        _check(lib().dbec_oracle_set_ramp(self._h, int(nstp), G0, D0, G1, D1), "set_ramp")

    def get_coupling(self):
        g, d = C.c_double(), C.c_double()
        _check(lib().dbec_oracle_get_coupling(self._h, C.byref(g), C.byref(d)), "get_coupling")
        return g.value, d.value

    def density_1d(self, axis) -> np.ndarray:
        n = (self.p.nx, self.p.ny, self.p.nz)[axis]
        out = np.empty(n, dtype=np.float64)
        _check(lib().dbec_oracle_density_1d(self._h, int(axis), _dp(out)), "density_1d")
        return out

    def density_2d(self, axis) -> np.ndarray:
        """axis = the integrated one; shape (nz, ny, nx) with that axis removed."""
        shp = [self.p.nz, self.p.ny, self.p.nx]
        del shp[2 - axis]
        out = np.empty(shp, dtype=np.float64)
        _check(lib().dbec_oracle_density_2d(self._h, int(axis), _dp(out)), "density_2d")
        return out

    def observables(self) -> dict:
        o = OracleObs()
        _check(lib().dbec_oracle_observables(self._h, C.byref(o)), "observables")
        return o.as_dict()


# ---- single parts ----

def fft(a, sign=-1, naive=False) -> np.ndarray:
    """Unscaled DFT over every axis of a (1-D, 2-D or 3-D complex array)."""
    b = _c128(a)
    shp = list(b.shape)
    while len(shp) < 3:
        shp.insert(0, 1)
    nz, ny, nx = shp
    _check(lib().dbec_oracle_fft(_dp(b), nx, ny, nz, sign, int(naive)), "fft")
    return b


def erfcx(x):
    return lib().dbec_oracle_erfcx(float(x))


def vdd3d(kx, ky, kz, cutoff=0.0):
    return lib().dbec_oracle_vdd3d(kx, ky, kz, cutoff)


def vdd2d(kx, ky, d_perp):
    return lib().dbec_oracle_vdd2d(kx, ky, d_perp)


def vdd2d_xz(kx, kz, d_perp):
    return lib().dbec_oracle_vdd2d_xz(kx, kz, d_perp)


def wavenumber(m, n, d):
    return lib().dbec_oracle_wavenumber(m, n, d)


def vdd_table(p: OracleParams) -> np.ndarray:
    shape = (p.nz, p.ny, p.nx) if p.ndim == 3 else (p.ny, p.nx)
    out = np.empty(shape, dtype=np.float64)
    _check(lib().dbec_oracle_vdd_table(C.byref(p), _dp(out)), "vdd_table")
    return out


def phi_dd(p: OracleParams, dens, naive=False) -> np.ndarray:
    d = np.ascontiguousarray(dens, dtype=np.float64)
    out = np.empty_like(d)
    _check(lib().dbec_oracle_phi_dd(C.byref(p), _dp(d), _dp(out), int(naive)), "phi_dd")
    return out


def nonlinear(p: OracleParams, psi, phi) -> np.ndarray:
    a = _c128(psi)
    f = np.ascontiguousarray(phi, dtype=np.float64)
    _check(lib().dbec_oracle_nonlinear(C.byref(p), _dp(a), _dp(f)), "nonlinear")
    return a


def cn_sweep(p: OracleParams, psi, axis) -> np.ndarray:
    a = _c128(psi)
    _check(lib().dbec_oracle_cn_sweep(C.byref(p), _dp(a), axis), "cn_sweep")
    return a


def cn_line(line, a: complex) -> np.ndarray:
    b = _c128(line)
    a = complex(a)
    _check(lib().dbec_oracle_cn_line(_dp(b), b.size, a.real, a.imag), "cn_line")
    return b


def normalize(p: OracleParams, psi) -> np.ndarray:
    a = _c128(psi)
    _check(lib().dbec_oracle_normalize(C.byref(p), _dp(a)), "normalize")
    return a


def norm(p: OracleParams, psi) -> float:
    a = _c128(psi)
    return lib().dbec_oracle_norm(C.byref(p), _dp(a))
