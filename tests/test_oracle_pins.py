"""Pins of the CPU oracle against what the mathematics fixes.

PAPER.md prints no formula and no number, so every pin is a closed form, an invariant, a dense /
brute-force solve on tiny inputs, or a library-routine restatement (numpy / scipy).  None of them
re-calls the oracle's own routine to produce the expected value.
"""
import math

import numpy as np
import pytest
import scipy.fft
import scipy.linalg
import scipy.special

from paper_1601_04640_b200.inputs import IMAG, REAL, Workload, axis_coords, initial_psi, random_psi, workload


def small3d(n=16, mode=IMAG, G=0.0, D=0.0, dx=0.5, dt=0.025, trap=(1.0, 1.0, 0.5), cutoff=0.0):
    return Workload("t", 3, n, n, n, dx, dx, dx, dt, *trap, G, D, G, D, mode, 1, 11, 1, cutoff=cutoff)


def small2d(n=32, mode=REAL, G=0.0, D=0.0, dx=0.25, dt=0.01, trap=(1.0, 1.5, 0.0)):
    return Workload("t", 2, n, n, 1, dx, dx, 1.0, dt, *trap, G, D, G, D, mode, 1, 12, 1)


# ------------------------------------------------------------------ P4: DFT
def test_fft_matches_bruteforce_dft_tiny(ob):
    rng = np.random.default_rng(0)
    a = rng.standard_normal((4, 8, 16)) + 1j * rng.standard_normal((4, 8, 16))
    # brute force straight from the definition, python-side
    nz, ny, nx = a.shape
    Wz = np.exp(-2j * np.pi * np.outer(np.arange(nz), np.arange(nz)) / nz)
    Wy = np.exp(-2j * np.pi * np.outer(np.arange(ny), np.arange(ny)) / ny)
    Wx = np.exp(-2j * np.pi * np.outer(np.arange(nx), np.arange(nx)) / nx)
    ref = np.einsum("ai,bj,ck,ijk->abc", Wz, Wy, Wx, a)
    for naive in (False, True):
        out = ob.fft(a, sign=-1, naive=naive)
        assert np.max(np.abs(out - ref)) / np.max(np.abs(ref)) < 1e-13
        back = ob.fft(out, sign=+1, naive=naive) / a.size
        assert np.max(np.abs(back - a)) < 1e-13


def test_fft_against_library_and_invariants(ob):
    rng = np.random.default_rng(1)
    a = rng.standard_normal((16, 32, 64)) + 1j * rng.standard_normal((16, 32, 64))
    out = ob.fft(a, -1)
    ref = scipy.fft.fftn(a)
    assert np.max(np.abs(out - ref)) / np.max(np.abs(ref)) < 1e-13
    inv = ob.fft(a, +1)
    assert np.max(np.abs(inv - scipy.fft.ifftn(a) * a.size)) / np.max(np.abs(inv)) < 1e-13
    # Parseval
    assert abs(np.sum(np.abs(out) ** 2) / a.size - np.sum(np.abs(a) ** 2)) < 1e-9 * np.sum(np.abs(a) ** 2)
    # delta <-> constant
    d = np.zeros((8, 8, 8), complex)
    d[0, 0, 0] = 1.0
    assert np.max(np.abs(ob.fft(d, -1) - 1.0)) < 1e-15
    # shifted delta -> pure phase with the forward sign convention exp(-2 pi i m j / N)
    d = np.zeros((1, 1, 16), complex)
    d[0, 0, 3] = 1.0
    ph = np.exp(-2j * np.pi * 3 * np.arange(16) / 16)
    assert np.max(np.abs(ob.fft(d, -1)[0, 0] - ph)) < 4e-15   # ph itself carries the rounding of its angle
    # real input -> Hermitian spectrum
    r = rng.standard_normal((8, 8, 16))
    R = ob.fft(r, -1)
    Rm = np.conj(R[(-np.arange(8)) % 8][:, (-np.arange(8)) % 8][:, :, (-np.arange(16)) % 16])
    assert np.max(np.abs(R - Rm)) < 1e-12


# ------------------------------------------------------------------ P3: Crank-Nicolson sweep
@pytest.mark.parametrize("a", [0.025, 0.125j, 0.4, 2.5j])
@pytest.mark.parametrize("N", [3, 4, 17, 64])
def test_cn_line_against_dense_solve(ob, a, N):
    rng = np.random.default_rng(N)
    psi = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    M = N - 2
    L = 2 * np.eye(M) - np.eye(M, k=1) - np.eye(M, k=-1)          # -delta^2 on the interior
    rhs = a * psi[:-2] + (1 - 2 * a) * psi[1:-1] + a * psi[2:]      # uses the actual end values
    ref = np.zeros(N, complex)
    ref[1:-1] = np.linalg.solve(np.eye(M) + a * L, rhs)
    out = ob.cn_line(psi, a)
    assert out[0] == 0 and out[-1] == 0
    assert np.max(np.abs(out - ref)) < 1e-14 * max(1.0, np.max(np.abs(ref)))


@pytest.mark.parametrize("a", [0.025, 0.125j])
def test_cn_line_sine_mode_closed_form(ob, a):
    N = 34
    M = N - 2
    j = np.arange(N)
    for m in (1, 2, 7, M):
        mode = np.sin(np.pi * j * m / (M + 1))
        mode[0] = mode[-1] = 0.0
        lam = 4 * np.sin(np.pi * m / (2 * (M + 1))) ** 2
        mult = (1 - a * lam) / (1 + a * lam)
        out = ob.cn_line(mode.astype(complex), a)
        assert np.max(np.abs(out - mult * mode)) < 5e-15
        if isinstance(a, complex):
            assert abs(abs(mult) - 1.0) < 1e-15                     # unitary in real time


def test_cn_sweeps_axes_strides_and_commutation(ob):
    w = Workload("t", 3, 8, 16, 32, 0.3, 0.4, 0.5, 0.02, 1, 1, 1, 0, 0, 0, 0, REAL, 1, 5, 1)
    p = ob.params_of(w)
    psi = random_psi(w, 3)
    # each axis sweep == the line solver applied along that numpy axis (numpy axis 2 is x)
    for axis, npax, h in ((0, 2, w.dx), (1, 1, w.dy), (2, 0, w.dz)):
        a = 1j * w.dt / (4 * h * h)
        N = psi.shape[npax]
        M = N - 2
        A = np.eye(M) * (1 + 2 * a) - a * (np.eye(M, k=1) + np.eye(M, k=-1))
        B = np.eye(M) * (1 - 2 * a) + a * (np.eye(M, k=1) + np.eye(M, k=-1))
        mv = np.moveaxis(psi, npax, 0)
        rhs = np.tensordot(B, mv[1:-1], axes=1)
        rhs[0] += a * mv[0]
        rhs[-1] += a * mv[-1]
        sol = np.linalg.solve(A, rhs.reshape(M, -1)).reshape(rhs.shape)
        ref = np.zeros_like(mv)
        ref[1:-1] = sol
        ref = np.moveaxis(ref, 0, npax)
        out = ob.cn_sweep(p, psi, axis)
        assert np.max(np.abs(out - ref)) < 1e-14
    # the three sweeps commute (constant coefficients, separable, Dirichlet)
    xyz = ob.cn_sweep(p, ob.cn_sweep(p, ob.cn_sweep(p, psi, 0), 1), 2)
    zyx = ob.cn_sweep(p, ob.cn_sweep(p, ob.cn_sweep(p, psi, 2), 1), 0)
    assert np.max(np.abs(xyz - zyx)) < 1e-15 * 10


def test_cn_real_time_conserves_plain_sum_norm(ob):
    w = small3d(16, REAL)
    p = ob.params_of(w)
    psi = random_psi(w, 9)
    for ax in range(3):                     # zero faces first so that the map is the Cayley transform
        psi = ob.cn_sweep(p, psi, ax)
    n0 = ob.norm(p, psi)
    out = psi
    for ax in range(3):
        out = ob.cn_sweep(p, out, ax)
    assert abs(ob.norm(p, out) / n0 - 1) < 1e-14


# ------------------------------------------------------------------ P6: dipolar kernels
def test_erfcx_against_scipy(ob):
    for x in [0.0, 1e-8, 0.3, 1.0, 2.999, 3.0, 3.001, 5.0, 10.0, 26.0, 27.0, 31.4, 100.0, 1e4]:
        ref = scipy.special.erfcx(x)
        assert abs(ob.erfcx(x) - ref) <= 2e-15 * ref + 1e-300, x


def test_vdd3d_properties(ob):
    assert ob.vdd3d(0, 0, 0) == 0.0
    assert ob.vdd3d(0, 0, 1.7) == pytest.approx(2.0, abs=1e-15)      # k along the dipoles
    assert ob.vdd3d(1.3, 0, 0) == pytest.approx(-1.0, abs=1e-15)     # k perpendicular
    assert ob.vdd3d(1.0, 1.0, 1.0) == pytest.approx(0.0, abs=1e-15)  # magic angle
    for s in ((-1, 1, 1), (1, -1, 1), (1, 1, -1)):
        assert ob.vdd3d(0.3 * s[0], 0.7 * s[1], 1.1 * s[2]) == ob.vdd3d(0.3, 0.7, 1.1)
    # depends on kx, ky only through kx^2 + ky^2
    assert ob.vdd3d(0.6, 0.8, 0.5) == pytest.approx(ob.vdd3d(1.0, 0.0, 0.5), abs=1e-15)
    w = small3d(16)
    V = ob.vdd_table(ob.params_of(w))
    assert V.min() >= -1 - 1e-15 and V.max() <= 2 + 1e-15
    assert V[0, 0, 0] == 0
    assert abs(V.sum()) < 1e-11                                      # cubic grid: angular average 0
    # index -> wavenumber map (S6): m and N-m give the same kernel; kz is numpy axis 0
    assert np.array_equal(V[1:, :, :], V[:0:-1, :, :])
    assert V[3, 0, 0] == pytest.approx(2.0) and V[0, 3, 0] == pytest.approx(-1.0) and V[0, 0, 3] == pytest.approx(-1.0)
    assert ob.wavenumber(1, 16, 0.5) == pytest.approx(2 * math.pi / 8)
    assert ob.wavenumber(15, 16, 0.5) == pytest.approx(-2 * math.pi / 8)


def test_vdd3d_cutoff_limits(ob):
    # kR -> infinity: untruncated kernel; kR -> 0: kernel vanishes like (kR)^2/10
    assert ob.vdd3d(0.3, 0.2, 0.9, 1e9) == pytest.approx(ob.vdd3d(0.3, 0.2, 0.9, 0.0), rel=1e-12)
    k = 0.1     # 1 + 3cos(x)/x^2 - 3sin(x)/x^3 = x^2/10 - x^4/280 + O(x^6)
    assert ob.vdd3d(0, 0, k, 1.0) == pytest.approx(2.0 * (k * k / 10.0 - k ** 4 / 280.0), rel=1e-6)


def test_vdd2d_properties(ob):
    assert ob.vdd2d(0, 0, 1.0) == 2.0
    xs = np.linspace(0, 60, 400)
    h = np.array([ob.vdd2d(x, 0.0, 1.0) for x in xs])
    assert np.all(np.diff(h) < 0)                                    # monotone decreasing
    assert np.all(np.isfinite(h))
    assert h[-1] > -1 and h[-1] == pytest.approx(-1.0, abs=2e-3)
    # isotropic in the plane; scales with d_perp
    assert ob.vdd2d(3, 4, 0.5) == pytest.approx(ob.vdd2d(5, 0, 0.5), abs=1e-15)
    assert ob.vdd2d(2.0, 0, 1.0) == pytest.approx(ob.vdd2d(1.0, 0, 2.0), abs=1e-15)
    # library value
    xi = 1.3 / math.sqrt(2)
    assert ob.vdd2d(1.3, 0, 1.0) == pytest.approx(2 - 3 * math.sqrt(math.pi) * xi * scipy.special.erfcx(xi), abs=1e-15)
    # = Gaussian average over k_z of the 3-D kernel (defining property of the quasi-2-D reduction)
    kz = np.linspace(-40, 40, 400001)
    wgt = np.exp(-kz ** 2 / 2.0) / math.sqrt(2 * math.pi)            # |FT of the d_perp=1 Gaussian density|
    kr = 1.3
    avg = np.trapezoid((3 * kz ** 2 / (kz ** 2 + kr ** 2) - 1) * wgt, kz)
    assert ob.vdd2d(kr, 0, 1.0) == pytest.approx(avg, abs=1e-9)


# ------------------------------------------------------------------ P7: whole dipolar path
def _f_dip(x):
    s = math.sqrt(1 - x * x)
    return (1 + 2 * x * x) / (1 - x * x) - 3 * x * x * math.atanh(s) / (1 - x * x) ** 1.5


def test_phi_dd_gaussian_dipolar_energy_closed_form(ob):
    # Gaussian with nu = lambda = 1, kappa = 1/2: dV sum Phi n = -f(kappa_g) prod sqrt(w_d / 2 pi),
    # kappa_g = l_perp / l_z = sqrt(kappa / nu)   (textbook dipolar energy of a Gaussian cloud)
    for n, R, tol in ((32, 6.0, 3e-5), (64, 12.0, 2e-7)):
        w = small3d(n, cutoff=R)
        p = ob.params_of(w)
        psi = initial_psi(w, noise=0.0).real
        dens = psi ** 2
        phi = ob.phi_dd(p, dens)
        e = w.cell_volume * np.sum(phi * dens)
        ref = -_f_dip(math.sqrt(0.5)) * math.sqrt(1 / (2 * math.pi)) ** 2 * math.sqrt(0.5 / (2 * math.pi))
        assert e == pytest.approx(ref, rel=tol)
        assert e < 0        # cloud elongated along the dipoles: net attraction


def test_phi_dd_bruteforce_equals_fft_and_is_real_linear(ob):
    w = small3d(8)
    p = ob.params_of(w)
    rng = np.random.default_rng(5)
    n1 = rng.random(w.shape)
    n2 = rng.random(w.shape)
    a = ob.phi_dd(p, n1, naive=False)
    b = ob.phi_dd(p, n1, naive=True)
    assert np.max(np.abs(a - b)) < 1e-13
    # library restatement
    V = ob.vdd_table(p)
    ref = np.real(scipy.fft.ifftn(V * scipy.fft.fftn(n1)))
    assert np.max(np.abs(a - ref)) < 1e-13
    # linear; a constant density gives Phi = V(0) * const = 0 in 3-D
    assert np.max(np.abs(ob.phi_dd(p, 2 * n1 + 3 * n2) - 2 * a - 3 * ob.phi_dd(p, n2))) < 1e-12
    assert np.max(np.abs(ob.phi_dd(p, np.full(w.shape, 0.7)))) < 1e-14
    # single plane wave cos(k.r): eigenfunction with eigenvalue V_dd(k)
    iz, iy, ix = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    m = (1, 2, 3)   # (mx, my, mz)
    wave = np.cos(2 * np.pi * (m[0] * ix + m[1] * iy + m[2] * iz) / 8)
    k = [2 * np.pi * mm / (8 * 0.5) for mm in m]
    lam = 3 * k[2] ** 2 / (k[0] ** 2 + k[1] ** 2 + k[2] ** 2) - 1
    assert np.max(np.abs(ob.phi_dd(p, wave) - lam * wave)) < 1e-13


def test_phi_dd_2d_constant_density(ob):
    w = small2d(16)
    p = ob.params_of(w)
    out = ob.phi_dd(p, np.full(w.shape, 0.25))
    assert np.max(np.abs(out - 2.0 * 0.25)) < 1e-14                  # h(0) = 2


# ------------------------------------------------------------------ P1: nonlinear step
def test_nonlinear_special_cases(ob):
    w = small3d(8, IMAG, G=3.0, D=2.0)
    psi = random_psi(w, 1)
    rng = np.random.default_rng(2)
    phi = rng.standard_normal(w.shape)
    out = ob.nonlinear(ob.params_of(w), psi, phi)
    # phase untouched in imaginary time; decay exponent at hand-computed points
    assert np.max(np.abs(np.angle(out * np.conj(psi)))) < 1e-15
    c = (4, 4, 4)                                                    # centre: V = 0
    u = w.dt * (w.G * abs(psi[c]) ** 2 + w.D * phi[c])
    assert abs(out[c]) == pytest.approx(abs(psi[c]) * math.exp(-u), rel=1e-15)
    q = (1, 6, 7)                                                    # (iz, iy, ix): z=-1.5, y=1, x=1.5
    V = 0.5 * (1.0 * 1.5 ** 2 + 1.0 * 1.0 ** 2 + 0.25 * 1.5 ** 2)
    u = w.dt * (V + w.G * abs(psi[q]) ** 2 + w.D * phi[q])
    assert abs(out[q]) == pytest.approx(abs(psi[q]) * math.exp(-u), rel=1e-15)
    # real time: modulus untouched, phase = -dt U; two steps of dt == one step of 2 dt
    wr = small3d(8, REAL, G=3.0, D=2.0)
    outr = ob.nonlinear(ob.params_of(wr), psi, phi)
    assert np.max(np.abs(np.abs(outr) - np.abs(psi)) / np.abs(psi)) < 1e-15
    assert np.angle(outr[q] / psi[q]) == pytest.approx(-u, abs=1e-15)
    twice = ob.nonlinear(ob.params_of(wr), outr, phi)
    from dataclasses import replace
    once2 = ob.nonlinear(ob.params_of(replace(wr, dt=2 * wr.dt)), psi, phi)
    assert np.max(np.abs(twice - once2)) < 1e-15


# ------------------------------------------------------------------ P5: observables on a sampled Gaussian
def test_observables_sampled_gaussian_closed_forms(ob):
    w = Workload("t", 3, 32, 32, 32, 0.5, 0.5, 0.5, 0.025, 1.0, 1.0, 0.5, 45.0, 0.0, 45.0, 0.0, IMAG, 1, 1, 1)
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(initial_psi(w, noise=0.0))
    r = o.observables()
    om = (1.0, 1.0, 0.5)
    d = (0.5, 0.5, 0.5)
    ekin = sum((1 - math.exp(-om[i] * d[i] ** 2 / 4)) / d[i] ** 2 for i in range(3))
    etr = sum(om) / 4
    ec = 45.0 * math.prod(math.sqrt(x / (2 * math.pi)) for x in om)
    assert r["norm"] == pytest.approx(1.0, abs=1e-14)
    assert r["mu"] == pytest.approx(ekin + etr + ec, rel=2e-8)          # E_c aliasing ~1e-8 at dx = 0.5
    assert r["energy"] == pytest.approx(ekin + etr + ec / 2, rel=2e-8)
    assert r["rms_x"] == pytest.approx(1 / math.sqrt(2.0), rel=1e-12)
    assert r["rms_z"] == pytest.approx(1.0, rel=1e-11)          # tail cut at |z| = 8: ~4e-12
    assert r["rms_r"] == pytest.approx(math.sqrt(0.5 + 0.5 + 1.0), rel=1e-11)
    assert r["density0"] == pytest.approx(math.prod(math.sqrt(x / math.pi) for x in om), rel=1e-14)
    assert r["density_max"] == r["density0"]
    # G = 0: kinetic and trap closed forms to round-off
    o.set_coupling(0.0, 0.0)
    r0 = o.observables()
    assert r0["mu"] == pytest.approx(ekin + etr, rel=1e-11)       # z tail cut: ~2e-12
    assert r0["energy"] == pytest.approx(r0["mu"], rel=1e-15)


def test_observables_dipolar_term_and_mu_energy_split(ob):
    w = small3d(32, IMAG, G=10.0, D=7.0, cutoff=6.0)
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(initial_psi(w, noise=0.0))
    full = o.observables()
    o.set_coupling(10.0, 0.0)
    nod = o.observables()
    ed = -_f_dip(math.sqrt(0.5)) * (1 / (2 * math.pi)) * math.sqrt(0.5 / (2 * math.pi)) * 7.0
    assert full["mu"] - nod["mu"] == pytest.approx(ed, rel=1e-4)
    assert full["energy"] - nod["energy"] == pytest.approx(ed / 2, rel=1e-4)


# ------------------------------------------------------------------ P2: whole imaginary-time loop
def _lowest_discrete_eig(n, d, omega):
    x = axis_coords(n, d)[1:-1]
    M = n - 2
    H = (np.eye(M) * 2 - np.eye(M, k=1) - np.eye(M, k=-1)) / (2 * d * d) + np.diag(0.5 * omega ** 2 * x ** 2)
    return np.linalg.eigvalsh(H)[0]


def test_imag_time_noninteracting_ground_state_energy(ob):
    exact = 2 * _lowest_discrete_eig(32, 0.5, 1.0) + _lowest_discrete_eig(32, 0.5, 0.5)
    assert exact == pytest.approx(1.25 - (1 + 1 + 0.25) * 0.25 / 32, abs=4e-4)   # continuum + O(dx^2)
    errs = []
    for dt, steps in ((0.025, 600), (0.0125, 1200)):
        w = Workload("t", 3, 32, 32, 32, 0.5, 0.5, 0.5, dt, 1.0, 1.0, 0.5, 0, 0, 0, 0, IMAG, steps, 1, 1)
        o = ob.Oracle(ob.params_of(w))
        o.set_psi(initial_psi(w))
        o.step(steps)
        r = o.observables()
        assert r["norm"] == pytest.approx(1.0, abs=1e-14)
        assert r["mu"] == pytest.approx(r["energy"], abs=1e-13)
        errs.append(r["mu"] - exact)
    assert 0 < errs[0] < 1.5e-4                      # O(dt^2) splitting bias, variational from above
    assert 3.5 < errs[0] / errs[1] < 4.5             # quarters when dt halves


# ------------------------------------------------------------------ P8: real time
def test_real_time_norm_and_energy_conservation_and_phase_sign(ob):
    w = Workload("t", 2, 64, 64, 1, 0.25, 0.25, 1.0, 0.005, 1.0, 1.5, 0.0, 20.0, 15.0, 20.0, 15.0, REAL, 1, 2, 1)
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(initial_psi(w))
    r0 = o.observables()
    o.step(100)
    r1 = o.observables()
    assert abs(r1["norm"] - 1) < 1e-14
    assert abs(r1["energy"] - r0["energy"]) < 2e-3 * abs(r0["energy"])
    assert abs(r1["rms_x"] - r0["rms_x"]) > 1e-3          # it does evolve
    # phase sign: a stationary state of the discrete problem turns as exp(-i mu t)
    wi = Workload("t", 2, 32, 32, 1, 0.4, 0.4, 1.0, 0.002, 1.0, 1.0, 0.0, 0, 0, 0, 0, IMAG, 1, 3, 1)
    oi = ob.Oracle(ob.params_of(wi))
    oi.set_psi(initial_psi(wi, noise=0.0))
    oi.step(3000)
    gs = oi.get_psi()
    mu = oi.observables()["mu"]
    from dataclasses import replace
    orr = ob.Oracle(ob.params_of(replace(wi, time_mode=REAL)))
    orr.set_psi(gs)
    orr.step(10)
    ph = np.vdot(gs, orr.get_psi())
    assert abs(abs(ph) * wi.cell_volume - 1) < 1e-6
    assert np.angle(ph) == pytest.approx(-mu * 10 * wi.dt, abs=1e-6)


# ------------------------------------------------------------------ P9: library restatement of one step
def _numpy_step(w, psi, G, D, V_dd):
    """numpy/scipy restatement: rfftn/irfftn, solve_banded, numpy sums."""
    n = np.abs(psi) ** 2
    axes = tuple(range(psi.ndim))
    half = V_dd[..., : w.nx // 2 + 1]
    phi = scipy.fft.irfftn(scipy.fft.rfftn(n, axes=axes) * half, s=psi.shape, axes=axes)
    x = axis_coords(w.nx, w.dx)
    y = axis_coords(w.ny, w.dy)
    if w.ndim == 3:
        z = axis_coords(w.nz, w.dz)
        V = 0.5 * (w.nu ** 2 * x[None, None, :] ** 2 + w.lam ** 2 * y[None, :, None] ** 2 + w.kappa ** 2 * z[:, None, None] ** 2)
    else:
        V = 0.5 * (w.nu ** 2 * x[None, :] ** 2 + w.lam ** 2 * y[:, None] ** 2)
    c = 1.0 if w.time_mode == IMAG else 1j
    psi = psi * np.exp(-c * w.dt * (V + G * n + D * phi))
    hs = (w.dx, w.dy, w.dz)
    for ax in range(w.ndim):
        npax = psi.ndim - 1 - ax
        a = c * w.dt / (4 * hs[ax] ** 2)
        mv = np.moveaxis(psi, npax, 0)
        N = mv.shape[0]
        rhs = a * mv[:-2] + (1 - 2 * a) * mv[1:-1] + a * mv[2:]
        ab = np.zeros((3, N - 2), dtype=complex)
        ab[0, 1:] = -a
        ab[1, :] = 1 + 2 * a
        ab[2, :-1] = -a
        sol = scipy.linalg.solve_banded((1, 1), ab, rhs.reshape(N - 2, -1)).reshape(rhs.shape)
        new = np.zeros_like(mv)
        new[1:-1] = sol
        psi = np.moveaxis(new, 0, npax)
    if w.time_mode == IMAG:
        psi = psi / np.sqrt(np.sum(np.abs(psi) ** 2) * w.cell_volume)
    return np.ascontiguousarray(psi)


@pytest.mark.parametrize("key,mode,steps", [("C1", IMAG, 3), ("C1", REAL, 3), ("2d", REAL, 3), ("2d", IMAG, 2), ("aniso", REAL, 2),
                                            ("2dxz", REAL, 3), ("2dxz", IMAG, 2)])
def test_full_step_against_numpy_scipy_restatement(ob, key, mode, steps):
    from dataclasses import replace
    if key == "C1":
        w = replace(workload("C1"), time_mode=mode)
    elif key == "2d":
        w = Workload("t", 2, 64, 32, 1, 0.2, 0.3, 1.0, 0.004, 1.0, 1.5, 0.0, 20.0, 15.0, 25.0, 15.0, mode, 1, 2, 1)
    elif key == "2dxz":
        w = Workload("t", 2, 32, 64, 1, 0.3, 0.2, 1.0, 0.004, 1.0, 0.7, 0.0, 20.0, 15.0, 25.0, 15.0, mode, 1, 2, 1,
                     d_perp=0.8, plane=1)
    else:
        w = Workload("t", 3, 16, 32, 8, 0.4, 0.3, 0.8, 0.01, 1.0, 1.2, 0.8, 50.0, 40.0, 50.0, 45.0, mode, 1, 4, 1)
    p = ob.params_of(w)
    o = ob.Oracle(p)
    psi = random_psi(w, 21) if mode == REAL else initial_psi(w)
    o.set_psi(psi)
    o.set_coupling(w.G_run, w.D_run)
    V_dd = _numpy_vdd(w)        # numpy.fft.fftfreq wavenumbers, scipy erfcx: nothing from the oracle
    ref = psi
    for _ in range(steps):
        ref = _numpy_step(w, ref, w.G_run, w.D_run, V_dd)
    o.step(steps)
    out = o.get_psi()
    assert np.max(np.abs(out - ref)) / np.max(np.abs(ref)) < 1e-13


def test_step_order_is_nonlinear_then_x_y_z_then_norm(ob):
    w = small3d(16, IMAG, G=20.0, D=10.0)
    p = ob.params_of(w)
    psi = initial_psi(w)
    o = ob.Oracle(p)
    o.set_psi(psi)
    o.step(1)
    phi = ob.phi_dd(p, np.abs(psi) ** 2)
    ref = ob.nonlinear(p, psi, phi)
    for ax in range(3):
        ref = ob.cn_sweep(p, ref, ax)
    ref = ob.normalize(p, ref)
    assert np.array_equal(o.get_psi(), ref)
    assert ob.norm(p, ref) == pytest.approx(1.0, abs=1e-15)


# ------------------------------------------------------------------ anisotropic spacings (dx != dy != dz)
# Every pin above that touches V_dd, dV, E_kin or rms uses a cubic grid; C5 (dz = 2 dx) and every 2-D
# run with dx != dy rest on the branches pinned here.  Expected values are computed in the test from
# k_d = 2 pi m_d / (N_d d_d) and from the closed forms of a sampled Gaussian, never from the oracle.
def _numpy_vdd(w):
    """V_dd on the full index grid from numpy.fft.fftfreq (readings S3, S4, S6, S21; no cutoff)."""
    kx = 2 * np.pi * np.fft.fftfreq(w.nx, w.dx)
    ky = 2 * np.pi * np.fft.fftfreq(w.ny, w.dy)
    if w.ndim == 2:
        xi = np.sqrt(kx[None, :] ** 2 + ky[:, None] ** 2) * w.d_perp / math.sqrt(2.0)
        if w.plane == 1:                                   # S25: second grid axis = polarisation axis z
            xiz = np.broadcast_to(ky[:, None] * w.d_perp / math.sqrt(2.0), xi.shape)
            with np.errstate(invalid="ignore", divide="ignore"):
                r = np.where(xi > 0, xiz ** 2 / xi, 0.0)
            return -1.0 + 3.0 * math.sqrt(math.pi) * r * scipy.special.erfcx(xi)
        return 2.0 - 3.0 * math.sqrt(math.pi) * xi * scipy.special.erfcx(xi)
    kz = 2 * np.pi * np.fft.fftfreq(w.nz, w.dz)
    KZ, KY, KX = np.meshgrid(kz, ky, kx, indexing="ij")
    k2 = KX ** 2 + KY ** 2 + KZ ** 2
    with np.errstate(invalid="ignore", divide="ignore"):
        v = np.where(k2 > 0, 3 * KZ ** 2 / k2 - 1, 0.0)
    return v


def test_phi_dd_plane_wave_eigenvalue_anisotropic_spacing(ob):
    nx, ny, nz = 8, 16, 4
    d = (0.5, 0.3, 0.8)
    w = Workload("t", 3, nx, ny, nz, *d, 0.01, 1, 1, 1, 0, 0, 0, 0, IMAG, 1, 1, 1)
    p = ob.params_of(w)
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    for m in ((1, 2, 1), (3, 0, 1), (0, 5, 1), (2, 3, 0), (1, 1, 1), (0, 0, 1), (3, 7, 1)):
        wave = np.cos(2 * np.pi * (m[0] * ix / nx + m[1] * iy / ny + m[2] * iz / nz))
        k = [2 * np.pi * m[i] / ((nx, ny, nz)[i] * d[i]) for i in range(3)]
        lam = 3 * k[2] ** 2 / (k[0] ** 2 + k[1] ** 2 + k[2] ** 2) - 1
        assert np.max(np.abs(ob.phi_dd(p, wave) - lam * wave)) < 1e-13, m
    # the whole table against numpy.fft.fftfreq wavenumbers
    assert np.max(np.abs(ob.vdd_table(p) - _numpy_vdd(w))) < 1e-14
    # 2-D, dx != dy: eigenvalue h(xi) with xi from both spacings
    w2 = Workload("t", 2, 16, 8, 1, 0.2, 0.35, 1.0, 0.01, 1, 1, 0, 0, 0, 0, 0, IMAG, 1, 1, 1, d_perp=0.7)
    p2 = ob.params_of(w2)
    jy, jx = np.meshgrid(np.arange(8), np.arange(16), indexing="ij")
    for m in ((1, 0), (0, 1), (3, 2), (5, 3)):
        wave = np.cos(2 * np.pi * (m[0] * jx / 16 + m[1] * jy / 8))
        kx, ky = 2 * np.pi * m[0] / (16 * 0.2), 2 * np.pi * m[1] / (8 * 0.35)
        xi = math.hypot(kx, ky) * 0.7 / math.sqrt(2)
        lam = 2 - 3 * math.sqrt(math.pi) * xi * scipy.special.erfcx(xi)
        assert np.max(np.abs(ob.phi_dd(p2, wave) - lam * wave)) < 1e-13, m
    assert np.max(np.abs(ob.vdd_table(p2) - _numpy_vdd(w2))) < 1e-14


def test_observables_sampled_gaussian_anisotropic_spacing(ob):
    om = (1.0, 1.3, 0.6)
    d = (0.5, 0.4, 0.25)
    G = 45.0
    w = Workload("t", 3, 32, 32, 64, *d, 0.01, *om, G, 0.0, G, 0.0, IMAG, 1, 1, 1)
    o = ob.Oracle(ob.params_of(w))
    x, y, z = axis_coords(32, d[0]), axis_coords(32, d[1]), axis_coords(64, d[2])
    # the analytic Gaussian itself, NOT normalised on the grid: norm = 1 only with dV = dx dy dz
    g = [(om[i] / math.pi) ** 0.25 * np.exp(-0.5 * om[i] * c * c) for i, c in enumerate((x, y, z))]
    psi = (g[2][:, None, None] * g[1][None, :, None] * g[0][None, None, :]).astype(complex)
    o.set_psi(psi)
    r = o.observables()
    ekin_d = [(1 - math.exp(-om[i] * d[i] ** 2 / 4)) / d[i] ** 2 for i in range(3)]
    etr = sum(om) / 4
    ec = G * math.prod(math.sqrt(v / (2 * math.pi)) for v in om)
    assert r["norm"] == pytest.approx(1.0, abs=1e-13)
    assert r["rms_x"] == pytest.approx(1 / math.sqrt(2 * om[0]), rel=1e-11)
    assert r["rms_y"] == pytest.approx(1 / math.sqrt(2 * om[1]), rel=1e-11)
    assert r["rms_z"] == pytest.approx(1 / math.sqrt(2 * om[2]), rel=1e-11)
    assert r["rms_r"] == pytest.approx(math.sqrt(sum(1 / (2 * v) for v in om)), rel=1e-11)
    assert r["density0"] == pytest.approx(math.prod(math.sqrt(v / math.pi) for v in om), rel=1e-14)
    assert r["mu"] == pytest.approx(sum(ekin_d) + etr + ec, rel=3e-8)        # E_c aliasing at dx = 0.5
    assert r["energy"] == pytest.approx(sum(ekin_d) + etr + ec / 2, rel=3e-8)
    o.set_coupling(0.0, 0.0)
    r0 = o.observables()
    assert r0["mu"] == pytest.approx(sum(ekin_d) + etr, rel=1e-11)
    # each kinetic term alone: a state flat along the other two axes is not available on a Dirichlet box,
    # so isolate an axis by differencing two trap-free evaluations with one spacing doubled in the CLOSED
    # FORM only: E_kin,z enters with 1/dz^2 — scaling psi's z-profile cannot mimic a wrong spacing
    for ax in range(3):
        om2 = list(om)
        om2[ax] *= 1.7                                                   # narrower along one axis only
        g2 = [(om2[i] / math.pi) ** 0.25 * np.exp(-0.5 * om2[i] * c * c) for i, c in enumerate((x, y, z))]
        o.set_psi((g2[2][:, None, None] * g2[1][None, :, None] * g2[0][None, None, :]).astype(complex))
        r2 = o.observables()
        dkin = (1 - math.exp(-om2[ax] * d[ax] ** 2 / 4)) / d[ax] ** 2 - ekin_d[ax]
        dtr = om[ax] ** 2 / (4 * om2[ax]) - om[ax] / 4                   # <x^2> = 1/(2 om2) in the same trap
        assert r2["mu"] - r0["mu"] == pytest.approx(dkin + dtr, rel=1e-8), ax   # aliasing e^{-pi^2/(om dx^2)} ~ 8e-11


def test_observables_2d_anisotropic_spacing(ob):
    om = (1.0, 1.5)
    d = (0.25, 0.4)
    w = Workload("t", 2, 64, 32, 1, d[0], d[1], 1.0, 0.01, om[0], om[1], 0.0, 0, 0, 0, 0, IMAG, 1, 1, 1)
    o = ob.Oracle(ob.params_of(w))
    x, y = axis_coords(64, d[0]), axis_coords(32, d[1])
    gx = (om[0] / math.pi) ** 0.25 * np.exp(-0.5 * om[0] * x * x)
    gy = (om[1] / math.pi) ** 0.25 * np.exp(-0.5 * om[1] * y * y)
    o.set_psi((gy[:, None] * gx[None, :]).astype(complex))
    r = o.observables()
    ekin = sum((1 - math.exp(-om[i] * d[i] ** 2 / 4)) / d[i] ** 2 for i in range(2))
    assert r["norm"] == pytest.approx(1.0, abs=1e-13)
    assert r["mu"] == pytest.approx(ekin + sum(om) / 4, rel=1e-11)
    assert r["rms_x"] == pytest.approx(1 / math.sqrt(2 * om[0]), rel=1e-11)
    assert r["rms_y"] == pytest.approx(1 / math.sqrt(2 * om[1]), rel=1e-11)
    assert r["rms_z"] == 0.0


def test_density_max_off_centre(ob):
    w = Workload("t", 3, 16, 8, 8, 0.5, 0.4, 0.3, 0.01, 1, 1, 1, 0, 0, 0, 0, IMAG, 1, 1, 1)
    psi = 0.1 * random_psi(w, 3)
    psi[5, 2, 11] = 3.0 - 4.0j                       # (iz, iy, ix), far from the centre index (4, 4, 8)
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(psi)
    r = o.observables()
    assert r["density_max"] == 25.0
    assert r["density0"] == pytest.approx(abs(psi[4, 4, 8]) ** 2, rel=1e-15)
    assert r["density0"] < 1.0


# ------------------------------------------------------------------ S25: 2-D XZ plane (in-plane dipoles)
def test_vdd2d_xz_properties(ob):
    sp = math.sqrt(math.pi)
    assert ob.vdd2d_xz(0, 0, 1.0) == -1.0                              # k = 0
    for kx in (0.1, 1.0, 7.0, 45.0):
        assert ob.vdd2d_xz(kx, 0.0, 1.0) == pytest.approx(-1.0, abs=1e-15)   # k perpendicular to the dipoles
    for kz in (1e-3, 0.3, 1.3, 5.0, 40.0, 90.0):                       # k along the dipoles: 1 - h(xi)
        xi = kz / math.sqrt(2)
        assert ob.vdd2d_xz(0.0, kz, 1.0) == pytest.approx(-1 + 3 * sp * xi * scipy.special.erfcx(xi), rel=1e-14)
        assert ob.vdd2d_xz(0.0, kz, 1.0) == pytest.approx(1 - ob.vdd2d(kz, 0.0, 1.0), abs=1e-14)
    assert ob.vdd2d_xz(0.0, 1e5, 1.0) == pytest.approx(2.0, abs=1e-9)  # sqrt(pi) xi erfcx(xi) -> 1
    # even in both components, scales with d_perp, NOT isotropic
    assert ob.vdd2d_xz(-0.7, 1.1, 0.9) == ob.vdd2d_xz(0.7, 1.1, 0.9) == ob.vdd2d_xz(0.7, -1.1, 0.9)
    assert ob.vdd2d_xz(2.0, 1.0, 1.0) == pytest.approx(ob.vdd2d_xz(1.0, 0.5, 2.0), abs=1e-15)
    assert abs(ob.vdd2d_xz(3.0, 4.0, 0.5) - ob.vdd2d_xz(4.0, 3.0, 0.5)) > 0.1
    # library value at a generic point
    kx, kz, d = 0.9, 1.7, 0.6
    xi, xiz = math.hypot(kx, kz) * d / math.sqrt(2), kz * d / math.sqrt(2)
    assert ob.vdd2d_xz(kx, kz, d) == pytest.approx(-1 + 3 * sp * xiz ** 2 / xi * scipy.special.erfcx(xi), rel=1e-14)
    # the dipolar tensor is traceless: polarisation along z (in plane) + along x (in plane: swap the
    # arguments) + along the frozen axis (the XY kernel h) sum to zero
    for kx, kz in ((0.3, 0.4), (2.0, 0.1), (11.0, 35.0)):
        tr = ob.vdd2d_xz(kx, kz, 1.0) + ob.vdd2d_xz(kz, kx, 1.0) + ob.vdd2d(kx, kz, 1.0)
        assert abs(tr) < 4e-15
    # defining property: the 3-D kernel (dipoles along z) averaged over k_y with the Gaussian weight of the
    # frozen direction
    ky = np.linspace(-40, 40, 400001)
    wgt = np.exp(-ky ** 2 / 2.0) / math.sqrt(2 * math.pi)
    for kx, kz in ((1.3, 0.0), (0.0, 1.3), (0.8, 1.9), (3.0, 0.5)):
        avg = np.trapezoid((3 * kz ** 2 / (kx ** 2 + ky ** 2 + kz ** 2) - 1) * wgt, ky)
        assert ob.vdd2d_xz(kx, kz, 1.0) == pytest.approx(avg, abs=1e-9)
    # large arguments stay finite (C2-sized grids reach xi ~ 31, where exp(xi^2) erfc(xi) is inf * 0)
    assert np.isfinite(ob.vdd2d_xz(30.0, 30.0, 1.0)) and -1 <= ob.vdd2d_xz(30.0, 30.0, 1.0) <= 2


def test_phi_dd_2d_xz_plane_waves_and_table(ob):
    w = Workload("t", 2, 16, 8, 1, 0.2, 0.35, 1.0, 0.01, 1, 1, 0, 0, 0, 0, 0, IMAG, 1, 1, 1, d_perp=0.7, plane=1)
    p = ob.params_of(w)
    assert p.plane == 1
    jy, jx = np.meshgrid(np.arange(8), np.arange(16), indexing="ij")
    for m in ((1, 0), (0, 1), (3, 2), (5, 3)):
        wave = np.cos(2 * np.pi * (m[0] * jx / 16 + m[1] * jy / 8))
        kx, kz = 2 * np.pi * m[0] / (16 * 0.2), 2 * np.pi * m[1] / (8 * 0.35)    # second grid axis = z
        xi, xiz = math.hypot(kx, kz) * 0.7 / math.sqrt(2), kz * 0.7 / math.sqrt(2)
        lam = -1 + 3 * math.sqrt(math.pi) * xiz ** 2 / xi * scipy.special.erfcx(xi)
        assert np.max(np.abs(ob.phi_dd(p, wave) - lam * wave)) < 1e-13, m
    assert np.max(np.abs(ob.vdd_table(p) - _numpy_vdd(w))) < 1e-14
    # a uniform density feels V(0) = -1 (XY: +2)
    assert np.max(np.abs(ob.phi_dd(p, np.full(w.shape, 0.25)) + 0.25)) < 1e-14
    # plane is rejected in 3-D and for values other than 0 / 1
    import ctypes as C
    bad = ob.params(3, 8, 8, 8, .5, .5, .5, .01, 1, 1, 1, 0, 0, 0, plane=1)
    h = C.c_void_p()
    assert ob.lib().dbec_oracle_create(C.byref(bad), C.byref(h)) != 0
    bad = ob.params(2, 8, 8, 1, .5, .5, .5, .01, 1, 1, 1, 0, 0, 0, plane=2)
    assert ob.lib().dbec_oracle_create(C.byref(bad), C.byref(h)) != 0


# ------------------------------------------------------------------ S26: NSTP ramp of the nonlinearity
@pytest.mark.parametrize("mode", [IMAG, REAL])
def test_ramp_schedule_equals_explicit_couplings(ob, mode):
    w = small3d(16, mode, G=0.0, D=0.0, dt=0.02)
    p = ob.params_of(w)
    psi0 = initial_psi(w)
    G0, D0, G1, D1, n = 2.0, 1.0, 30.0, 18.0, 5
    a = ob.Oracle(p)
    a.set_psi(psi0)
    a.set_ramp(n, G0, D0, G1, D1)
    assert a.get_coupling() == (G0, D0)                # nothing has run yet
    b = ob.Oracle(p)
    b.set_psi(psi0)
    for k in range(1, n + 4):
        a.step(1)
        f = min(k, n) / n                              # the schedule written out here, not taken from the oracle
        b.set_coupling(G0 + (G1 - G0) * f, D0 + (D1 - D0) * f)
        b.step(1)
        assert a.get_coupling() == pytest.approx((G0 + (G1 - G0) * f, D0 + (D1 - D0) * f), rel=1e-15)
        assert np.array_equal(a.get_psi(), b.get_psi()), k
    assert a.get_coupling() == (G1, D1)                # exactly the end values once the ramp is over
    # first ramp step is NOT at the start value: step 1 of n runs with G0 + (G1 - G0)/n
    c = ob.Oracle(p)
    c.set_psi(psi0)
    c.set_coupling(G0, D0)
    c.step(1)
    d = ob.Oracle(p)
    d.set_psi(psi0)
    d.set_ramp(n, G0, D0, G1, D1)
    d.step(1)
    assert not np.array_equal(c.get_psi(), d.get_psi())
    # nstp = 0: end values at once; set_coupling cancels a running ramp
    e = ob.Oracle(p)
    e.set_ramp(0, G0, D0, G1, D1)
    assert e.get_coupling() == (G1, D1)
    e.set_ramp(4, 0.0, 0.0, 8.0, 4.0)
    e.set_psi(psi0)
    e.step(1)
    assert e.get_coupling() == (2.0, 1.0)
    e.set_coupling(5.0, 5.0)
    e.step(3)
    assert e.get_coupling() == (5.0, 5.0)


# ------------------------------------------------------------------ S27: integrated densities
def test_integrated_densities_closed_form_and_numpy(ob):
    om = (1.0, 1.3, 0.6)
    d = (0.5, 0.4, 0.25)
    w = Workload("t", 3, 32, 32, 64, *d, 0.01, *om, 0, 0, 0, 0, IMAG, 1, 1, 1)
    o = ob.Oracle(ob.params_of(w))
    cs = [axis_coords(n, dd) for n, dd in zip((32, 32, 64), d)]
    g = [(om[i] / math.pi) ** 0.25 * np.exp(-0.5 * om[i] * c * c) for i, c in enumerate(cs)]
    o.set_psi((g[2][:, None, None] * g[1][None, :, None] * g[0][None, None, :]).astype(complex))
    # marginals of a product Gaussian: sqrt(om/pi) exp(-om x^2) (the sampled sums over the other axes are 1
    # to ~1e-14, see test_observables_sampled_gaussian_anisotropic_spacing)
    for ax in range(3):
        n1 = o.density_1d(ax)
        ref = math.sqrt(om[ax] / math.pi) * np.exp(-om[ax] * cs[ax] ** 2)
        assert np.max(np.abs(n1 - ref)) < 1e-13, ax
        assert np.sum(n1) * d[ax] == pytest.approx(1.0, abs=1e-13)
    for ax in range(3):
        n2 = o.density_2d(ax)
        lo, hi = [b for b in range(3) if b != ax]
        ref = np.outer(math.sqrt(om[hi] / math.pi) * np.exp(-om[hi] * cs[hi] ** 2),
                       math.sqrt(om[lo] / math.pi) * np.exp(-om[lo] * cs[lo] ** 2))      # [hi][lo], lower axis fastest
        assert n2.shape == ref.shape
        assert np.max(np.abs(n2 - ref)) < 1e-13, ax
    # a rough complex field: numpy sums with each axis' own spacing
    wr = Workload("t", 3, 16, 8, 32, 0.3, 0.5, 0.7, 0.01, 1, 1, 1, 0, 0, 0, 0, REAL, 1, 1, 1)
    psi = random_psi(wr, 4)
    o2 = ob.Oracle(ob.params_of(wr))
    o2.set_psi(psi)
    n = np.abs(psi) ** 2                                              # [z][y][x]
    assert np.allclose(o2.density_1d(0), n.sum(axis=(0, 1)) * 0.5 * 0.7, rtol=1e-13, atol=0)
    assert np.allclose(o2.density_1d(1), n.sum(axis=(0, 2)) * 0.3 * 0.7, rtol=1e-13, atol=0)
    assert np.allclose(o2.density_1d(2), n.sum(axis=(1, 2)) * 0.3 * 0.5, rtol=1e-13, atol=0)
    assert np.allclose(o2.density_2d(2), n.sum(axis=0) * 0.7, rtol=1e-13, atol=0)
    assert np.allclose(o2.density_2d(1), n.sum(axis=1) * 0.5, rtol=1e-13, atol=0)
    assert np.allclose(o2.density_2d(0), n.sum(axis=2) * 0.3, rtol=1e-13, atol=0)
    # 2-D problem: 1-D densities only, weights dx / dy alone
    w2 = Workload("t", 2, 32, 16, 1, 0.2, 0.35, 1.0, 0.01, 1, 1, 0, 0, 0, 0, 0, REAL, 1, 1, 1)
    p2 = random_psi(w2, 5)
    o3 = ob.Oracle(ob.params_of(w2))
    o3.set_psi(p2)
    assert np.allclose(o3.density_1d(0), (np.abs(p2) ** 2).sum(axis=0) * 0.35, rtol=1e-13, atol=0)
    assert np.allclose(o3.density_1d(1), (np.abs(p2) ** 2).sum(axis=1) * 0.2, rtol=1e-13, atol=0)
    with pytest.raises(RuntimeError):
        o3.density_1d(2)
    with pytest.raises(RuntimeError):
        o3.density_2d(2)


# ------------------------------------------------------------------ f2: lengths that are not powers of two
@pytest.mark.parametrize("shape", [(1, 1, 6), (1, 1, 7), (1, 1, 15), (1, 1, 21), (1, 1, 35), (1, 1, 49), (1, 1, 50), (1, 1, 96),
                                   (1, 1, 210), (1, 1, 97), (3, 5, 7), (6, 10, 12), (12, 20, 48)])
def test_fft_any_length_matches_definition_and_library(ob, shape):
    rng = np.random.default_rng(sum(shape))
    a = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    out = ob.fft(a, -1)
    assert np.max(np.abs(out - scipy.fft.fftn(a))) / np.max(np.abs(out)) < 2e-14
    assert np.max(np.abs(ob.fft(a, +1) - scipy.fft.ifftn(a) * a.size)) / np.max(np.abs(out)) < 2e-14
    if a.size <= 5000:                                            # the O(N^2) definition (long double accumulation)
        assert np.max(np.abs(out - ob.fft(a, -1, naive=True))) / np.max(np.abs(out)) < 2e-14
    back = ob.fft(out, +1) / a.size
    assert np.max(np.abs(back - a)) < 1e-13


@pytest.mark.parametrize("mode", [IMAG, REAL])
def test_full_step_on_a_non_power_of_two_grid_against_numpy(ob, mode):
    w = Workload("t", 3, 12, 10, 6, 0.4, 0.3, 0.8, 0.01, 1.0, 1.2, 0.8, 50.0, 40.0, 50.0, 45.0, mode, 1, 4, 1)
    p = ob.params_of(w)
    o = ob.Oracle(p)
    psi = random_psi(w, 21) if mode == REAL else initial_psi(w)
    o.set_psi(psi)
    o.set_coupling(w.G_run, w.D_run)
    ref = psi
    for _ in range(2):
        ref = _numpy_step(w, ref, w.G_run, w.D_run, _numpy_vdd(w))
    o.step(2)
    assert np.max(np.abs(o.get_psi() - ref)) / np.max(np.abs(ref)) < 1e-13
    w2 = Workload("t", 2, 50, 14, 1, 0.2, 0.3, 1.0, 0.004, 1.0, 1.5, 0.0, 20.0, 15.0, 25.0, 15.0, mode, 1, 2, 1, plane=1)
    o2 = ob.Oracle(ob.params_of(w2))
    psi2 = random_psi(w2, 5)
    o2.set_psi(psi2)
    o2.set_coupling(w2.G_run, w2.D_run)
    o2.step(1)
    assert np.max(np.abs(o2.get_psi() - _numpy_step(w2, psi2, w2.G_run, w2.D_run, _numpy_vdd(w2)))) < 1e-13
