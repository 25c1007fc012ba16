"""Seeded synthetic inputs for the dipolar SSCN step (serves the tests, bench.py and smoke()).

This module holds NONE of the method's arithmetic: it only names the five workloads of
BASELINE.json (`configs`, restated in DESIGN.md "Input recipe") and draws the initial wave
function (reading S22): a normalised anisotropic Gaussian matching the trap plus 1e-3 uniform real
noise from a counter-based splitmix64 hash, faces zeroed, normalised with the plain sum x dV.
Both the CUDA path and the CPU oracle receive the array produced here; neither imports the other.

The paper's own example inputs are not available; these stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
import numpy as np

IMAG, REAL = 0, 1


@dataclass(frozen=True)
class Workload:
    name: str
    ndim: int
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    dt: float
    nu: float
    lam: float
    kappa: float
    G: float          # value the handle is created with
    D: float
    G_run: float      # value set with set_coupling before the first step (S18); == G if no quench
    D_run: float
    time_mode: int
    steps: int
    seed: int
    report_every: int
    d_perp: float = 1.0
    cutoff: float = 0.0
    plane: int = 0    # 2-D only: 0 = XY, 1 = XZ (the second grid axis ny/dy/lam is then the polarisation axis z)

    @property
    def shape(self):
        """numpy shape, slowest axis first; idx = ix + NX*(iy + NY*iz)."""
        return (self.nz, self.ny, self.nx) if self.ndim == 3 else (self.ny, self.nx)

    @property
    def npoints(self):
        return self.nx * self.ny * self.nz

    @property
    def cell_volume(self):
        return self.dx * self.dy * (self.dz if self.ndim == 3 else 1.0)


def _w(name, ndim, n, d, dt, trap, G, D, mode, steps, seed, every, G_run=None, D_run=None, plane=0):
    nx, ny, nz = n
    dx, dy, dz = d
    nu, lam, kappa = trap
    return Workload(name, ndim, nx, ny, nz, dx, dy, dz, dt, nu, lam, kappa, G, D,
                    G if G_run is None else G_run, D if D_run is None else D_run,
                    mode, steps, seed, every, plane=plane)


# BASELINE.json `configs`, in order.
WORKLOADS = {
    "C1": _w("imag3d_tiny_32", 3, (32, 32, 32), (0.5, 0.5, 0.5), 0.1 * 0.5 ** 2, (1.0, 1.0, 0.5),
             45.0, 30.0, IMAG, 300, 1, 100),
    "C2": _w("real2dXY_512", 2, (512, 512, 1), (0.1, 0.1, 1.0), 0.5 * 0.1 ** 2, (1.0, 1.5, 0.0),
             20.0, 15.0, REAL, 1000, 2, 250, G_run=25.0),
    "C3": _w("imag3d_mid_128", 3, (128, 128, 128), (0.2, 0.2, 0.2), 0.1 * 0.2 ** 2, (1.0, 1.0, 0.5),
             100.0, 80.0, IMAG, 2000, 3, 100),
    "C4": _w("real3d_256", 3, (256, 256, 256), (0.1, 0.1, 0.1), 0.5 * 0.1 ** 2, (1.0, 1.2, 0.8),
             200.0, 150.0, REAL, 500, 4, 50, D_run=180.0),
    "C5": _w("imag3d_cigar_512x512x256", 3, (512, 512, 256), (0.08, 0.08, 0.16), 0.05 * 0.08 ** 2,
             (1.0, 1.0, 0.25), 400.0, 350.0, IMAG, 200, 5, 200),
    # Not BASELINE.json configs: the three program variants of PAPER.md:15 that C1-C5 leave out (imag2dXY,
    # imag2dXZ, real2dXZ), so that all six (ndim, plane, time mode) combinations have a full-run golden file.
    # In the XZ plane the second grid axis (ny, dy, lam) is the polarisation axis z (reading S25).
    "X0": _w("imag2dXY_256", 2, (256, 256, 1), (0.15, 0.15, 1.0), 0.1 * 0.15 ** 2, (1.0, 1.5, 0.0),
             30.0, 20.0, IMAG, 600, 6, 200),
    "X1": _w("imag2dXZ_256x128", 2, (256, 128, 1), (0.15, 0.2, 1.0), 0.1 * 0.15 ** 2, (1.0, 0.6, 0.0),
             30.0, 15.0, IMAG, 600, 7, 200, plane=1),
    "X2": _w("real2dXZ_512", 2, (512, 512, 1), (0.1, 0.1, 1.0), 0.5 * 0.1 ** 2, (1.0, 0.8, 0.0),
             20.0, 12.0, REAL, 500, 8, 250, G_run=25.0, plane=1),
}


def workload(key: str, **overrides) -> Workload:
    w = WORKLOADS[key]
    return replace(w, **overrides) if overrides else w


_GOLDEN = np.uint64(0x9E3779B97F4A7C15)


def hash_uniform(seed: int, idx: np.ndarray) -> np.ndarray:
    """u(idx) in [0,1): splitmix64 finaliser of seed + (idx+1)*0x9E3779B97F4A7C15, top 53 bits."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + (idx.astype(np.uint64) + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def axis_coords(n: int, d: float) -> np.ndarray:
    """Grid coordinates of one axis, centre at index n//2 (reading S17)."""
    return (np.arange(n, dtype=np.float64) - (n // 2)) * d


def initial_psi(w: Workload, noise: float = 1e-3) -> np.ndarray:
    """complex128 array of shape w.shape (reading S22)."""
    x = axis_coords(w.nx, w.dx)
    y = axis_coords(w.ny, w.dy)
    gx = (w.nu / np.pi) ** 0.25 * np.exp(-0.5 * w.nu * x * x)
    gy = (w.lam / np.pi) ** 0.25 * np.exp(-0.5 * w.lam * y * y)
    if w.ndim == 3:
        z = axis_coords(w.nz, w.dz)
        gz = (w.kappa / np.pi) ** 0.25 * np.exp(-0.5 * w.kappa * z * z)
        re = gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
    else:
        re = gy[:, None] * gx[None, :]
    re = np.ascontiguousarray(re)
    flat = re.reshape(-1)
    chunk = 1 << 22
    for s in range(0, flat.size, chunk):
        e = min(flat.size, s + chunk)
        u = hash_uniform(w.seed, np.arange(s, e, dtype=np.uint64))
        flat[s:e] += noise * (2.0 * u - 1.0)
    # faces zeroed
    for ax in range(re.ndim):
        sl = [slice(None)] * re.ndim
        sl[ax] = 0
        re[tuple(sl)] = 0.0
        sl[ax] = -1
        re[tuple(sl)] = 0.0
    s = float(np.sum(re * re)) * w.cell_volume
    re /= np.sqrt(s)
    return re.astype(np.complex128)


def random_psi(w: Workload, seed: int) -> np.ndarray:
    """Rough complex test field (both parts non-zero): Gaussian envelope x complex hash noise."""
    base = initial_psi(w, noise=0.0).real
    idx = np.arange(base.size, dtype=np.uint64)
    a = hash_uniform(seed, idx).reshape(base.shape)
    b = hash_uniform(seed + 7919, idx).reshape(base.shape)
    psi = base * (0.5 + a) * np.exp(2j * np.pi * b)
    psi += 1e-3 * ((2 * hash_uniform(seed + 1, idx).reshape(base.shape) - 1)
                   + 1j * (2 * hash_uniform(seed + 2, idx).reshape(base.shape) - 1))
    s = float(np.sum(np.abs(psi) ** 2)) * w.cell_volume
    return (psi / np.sqrt(s)).astype(np.complex128)
