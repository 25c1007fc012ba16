"""GPU parity: the CUDA path (through the C ABI of include/dbec.h) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances: BASELINE.json `north_star` — psi after one step
within 1e-12 relative max-abs; mu, energy, rms within 1e-9 relative.  Single parts use the same
1e-12 bar.
"""
import json
import os

import numpy as np
import pytest

from paper_1601_04640_b200.inputs import IMAG, REAL, Workload, initial_psi, random_psi, workload

pytestmark = pytest.mark.gpu

PSI_TOL = 1e-12
OBS_TOL = 1e-9


@pytest.fixture(scope="module")
def gp():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1601_04640_b200 import dbec
    dbec.lib()
    return dbec


def relerr(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def grid3(nx, ny, nz, mode, G=30.0, D=20.0, dx=0.4, dt=None, trap=(1.0, 1.2, 0.7), cutoff=0.0, d=None):
    d = d or (dx, dx, dx)
    dt = dt if dt is not None else (0.1 if mode == IMAG else 0.5) * d[0] ** 2
    return Workload("t3", 3, nx, ny, nz, d[0], d[1], d[2], dt, *trap, G, D, G, D, mode, 1, 21, 1, cutoff=cutoff)


def grid2(nx, ny, mode, G=20.0, D=15.0, dx=0.2, dt=None, trap=(1.0, 1.5, 0.0), dy=None, plane=0):
    dt = dt if dt is not None else (0.1 if mode == IMAG else 0.5) * dx ** 2
    return Workload("t2", 2, nx, ny, 1, dx, dy or dx, 1.0, dt, *trap, G, D, G, D, mode, 1, 22, 1, plane=plane)


SHAPES3 = [(16, 16, 16), (32, 32, 32), (64, 16, 32), (16, 64, 128), (128, 32, 16), (256, 16, 16), (16, 256, 32),
           (32, 16, 512), (512, 32, 16)]
SHAPES2 = [(16, 16), (32, 64), (128, 32), (512, 16), (16, 512), (256, 256)]
# dx != dy != dz (C5 is the only BASELINE.json config with two spacings): the V_dd wavenumbers, dV, the
# Crank-Nicolson coefficient of every axis and the kinetic / rms sums each take their own spacing
ANISO3 = [(32, 16, 64), (128, 32, 16), (16, 128, 128)]
ANISO2 = [(64, 32), (128, 256)]
# 2-D XZ plane (in-plane dipoles, reading S25; PAPER.md:15 imag2dXZ / real2dXZ): same kernels, another V_dd table
XZ2 = [(32, 64), (256, 128), (512, 512)]


def all_small_workloads():
    out = []
    for mode in (IMAG, REAL):
        for s in SHAPES3:
            out.append(grid3(*s, mode))
        for s in SHAPES2:
            out.append(grid2(*s, mode))
        for s in ANISO3:
            out.append(grid3(*s, mode, d=(0.4, 0.3, 0.6)))
        for s in ANISO2:
            out.append(grid2(*s, mode, dx=0.2, dy=0.3))
        for s in XZ2:
            out.append(grid2(*s, mode, dx=0.2, dy=0.25, plane=1))
    return out


def wid(w):
    aniso = "" if (w.dx == w.dy and (w.ndim == 2 or w.dx == w.dz)) else "-aniso"
    return f"{w.ndim}d{'xz' if w.plane else ''}-{w.nx}x{w.ny}x{w.nz}-{'imag' if w.time_mode == IMAG else 'real'}{aniso}"


@pytest.mark.parametrize("w", all_small_workloads(), ids=wid)
def test_cn_sweeps_match_oracle(gp, ob, w):
    psi0 = random_psi(w, 5)
    sim = gp.Dbec(gp.params_of(w))
    for axis in range(w.ndim):
        sim.set_psi(psi0)
        sim.cn_sweep(axis)
        got = sim.get_psi()
        ref = ob.cn_sweep(ob.params_of(w), psi0, axis)
        assert relerr(got, ref) < PSI_TOL, f"axis {axis}"
    sim.close()


@pytest.mark.parametrize("w", all_small_workloads()[::2] + [grid3(32, 32, 32, IMAG, cutoff=5.0)], ids=wid)
def test_phi_dd_matches_oracle(gp, ob, w):
    psi0 = random_psi(w, 6)
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(psi0)
    got = sim.phi_dd().cpu().numpy()
    ref = ob.phi_dd(ob.params_of(w), np.abs(psi0) ** 2)
    assert relerr(got, ref) < PSI_TOL
    sim.close()


@pytest.mark.parametrize("w", all_small_workloads()[1::3], ids=wid)
def test_nonlinear_matches_oracle(gp, ob, w):
    psi0 = random_psi(w, 7)
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(psi0)
    sim.nonlinear()
    got = sim.get_psi()
    p = ob.params_of(w)
    ref = ob.nonlinear(p, psi0, ob.phi_dd(p, np.abs(psi0) ** 2))
    assert relerr(got, ref) < PSI_TOL
    sim.close()


def test_normalize_matches_oracle(gp, ob):
    w = grid3(32, 16, 64, IMAG)
    psi0 = 1.7 * random_psi(w, 8)
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(psi0)
    sim.normalize()
    got = sim.get_psi()
    ref = ob.normalize(ob.params_of(w), psi0)
    assert relerr(got, ref) < PSI_TOL
    assert abs(sim.observables()["norm"] - 1.0) < 1e-13
    sim.close()


def test_normalize_in_real_time_is_applied_once(gp, ob):
    """Real time never rewrites the deferred norm factor: dbec_normalize must apply it at once, or every
    later step multiplies psi by it again (round-1 advisor finding)."""
    w = grid3(32, 16, 64, REAL)
    psi0 = 1.7 * random_psi(w, 8)
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(psi0)
    sim.normalize()
    assert relerr(sim.get_psi(), ob.normalize(ob.params_of(w), psi0)) < PSI_TOL
    sim.step(3)
    got = sim.get_psi()
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(ob.normalize(ob.params_of(w), psi0))
    o.step(3)
    assert relerr(got, o.get_psi()) < PSI_TOL
    assert abs(sim.observables()["norm"] - o.observables()["norm"]) < 1e-13
    sim.close()
    o.close()


@pytest.mark.parametrize("shape", [(32, 32, 32), (128, 16, 16)])
def test_nonlinear_after_imaginary_time_steps(gp, ob, shape):
    """After an imaginary-time step the stored field carries a deferred factor s != 1; dbec_nonlinear must
    not apply it twice (round-1 advisor finding)."""
    w = grid3(*shape, IMAG)
    psi0 = 1.3 * initial_psi(w)
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(psi0)
    sim.step(2)
    sim.nonlinear()
    got = sim.get_psi()
    p = ob.params_of(w)
    o = ob.Oracle(p)
    o.set_psi(psi0)
    o.step(2)
    mid = o.get_psi()
    ref = ob.nonlinear(p, mid, ob.phi_dd(p, np.abs(mid) ** 2))
    assert relerr(got, ref) < PSI_TOL
    a = sim.observables()["norm"]
    assert abs(a - ob.norm(p, ref)) < 1e-12
    sim.close()
    o.close()


def test_device_pointer_psi_and_foreign_stream(gp, ob):
    """dbec_set_psi / dbec_get_psi with DEVICE pointers (the hand-off between handles) on a handle whose
    stream is not torch's current one, driven straight through the C ABI."""
    import ctypes as C
    import torch
    w = grid3(64, 32, 16, REAL)
    psi0 = random_psi(w, 4)
    side = torch.cuda.Stream()
    sim = gp.Dbec(gp.params_of(w), stream=side)
    d_in = torch.from_numpy(psi0).cuda()
    d_out = torch.empty_like(d_in)
    torch.cuda.synchronize()
    L = gp.lib()
    assert L.dbec_set_psi(sim._h, C.c_void_p(d_in.data_ptr()), 1) == 0
    assert L.dbec_step(sim._h, 2) == 0
    assert L.dbec_get_psi(sim._h, C.c_void_p(d_out.data_ptr()), 1) == 0
    side.synchronize()
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(psi0)
    o.step(2)
    assert relerr(d_out.cpu().numpy(), o.get_psi()) < PSI_TOL
    sim.close()
    o.close()


def one_step_pair(gp, ob, w, psi0, steps=1):
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(psi0)
    if (w.G_run, w.D_run) != (w.G, w.D):
        sim.set_coupling(w.G_run, w.D_run)
    sim.step(steps)
    got = sim.get_psi()
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(psi0)
    if (w.G_run, w.D_run) != (w.G, w.D):
        o.set_coupling(w.G_run, w.D_run)
    o.step(steps)
    ref = o.get_psi()
    return sim, o, got, ref


# shapes kernels_small_p2.cu is compiled for (the one-launch step with compile-time power-of-two lengths)
P2_SHAPES = [(a, b, c) for a in (16, 32, 64) for b in (16, 32, 64) for c in (16, 32, 64) if a * b * c <= 131072]


def small_step_cases():
    """(workload, cluster): "auto" = small 3-D grids take the one-launch cluster step (kernels_small.cu), everything
    else the multi-launch path; "0" = the multi-launch path also on the grids "auto" gives to the cluster step."""
    out = []
    for w in all_small_workloads():
        out.append((w, "auto"))
        if w.ndim == 3 and w.npoints <= 65536:
            out.append((w, "0"))
            if (w.nx, w.ny, w.nz) in P2_SHAPES:
                out.append((w, "general"))      # "auto" is k_small_p2 there: this one is k_small_step
    return out


@pytest.mark.parametrize("w,cluster", small_step_cases(), ids=lambda v: wid(v) if isinstance(v, Workload) else f"cluster-{v}")
def test_one_step_small_grids(gp, ob, w, cluster, monkeypatch):
    if cluster == "0":
        monkeypatch.setenv("DBEC_CLUSTER", "0")
    if cluster == "general":
        monkeypatch.setenv("DBEC_SMALL_P2", "0")
    psi0 = random_psi(w, 9) if w.time_mode == REAL else initial_psi(w)
    sim, o, got, ref = one_step_pair(gp, ob, w, psi0)
    if cluster != "0" and (w.nx, w.ny, w.nz) in P2_SHAPES:
        assert sim.pass_kernels() == {"sscn_step<cluster>": "k_small_step" if cluster == "general" else "k_small_p2"}
    assert relerr(got, ref) < PSI_TOL
    a, b = sim.observables(), o.observables()
    for k in b:
        if w.ndim == 2 and k == "rms_z":
            continue
        assert abs(a[k] - b[k]) <= OBS_TOL * max(abs(b[k]), 1e-300), k
    sim.close()
    o.close()


@pytest.mark.parametrize("key", ["C1", "C2", "C3", "C4", "C5"])
def test_one_step_baseline_configs(gp, ob, key):
    """Full-size BASELINE.json configs, one step, every grid point compared."""
    w = workload(key)
    psi0 = initial_psi(w)
    sim, o, got, ref = one_step_pair(gp, ob, w, psi0)
    assert relerr(got, ref) < PSI_TOL
    a, b = sim.observables(), o.observables()
    for k in ("norm", "mu", "energy", "rms_x", "rms_y", "rms_z", "rms_r", "density0", "density_max"):
        if w.ndim == 2 and k == "rms_z":
            continue
        assert abs(a[k] - b[k]) <= OBS_TOL * abs(b[k]), k
    sim.close()
    o.close()


def test_fused_and_unfused_x_sweep_agree(gp, monkeypatch):
    w = workload("C1")
    psi0 = initial_psi(w)
    outs = []
    monkeypatch.setenv("DBEC_CLUSTER", "0")            # the multi-launch path (C1 would take the one-launch step)
    for fuse in ("1", "0"):
        monkeypatch.setenv("DBEC_FUSE_CNX", fuse)
        sim = gp.Dbec(gp.params_of(w))
        sim.set_psi(psi0)
        sim.step(3)
        outs.append(sim.get_psi())
        sim.close()
    assert relerr(outs[0], outs[1]) < PSI_TOL


def test_graph_and_plain_launches_agree_bitwise(gp, monkeypatch):
    w = workload("C1")
    psi0 = initial_psi(w)
    outs = []
    monkeypatch.setenv("DBEC_CLUSTER", "0")
    for g in ("1", "0"):
        monkeypatch.setenv("DBEC_GRAPH", g)
        sim = gp.Dbec(gp.params_of(w))
        sim.set_psi(psi0)
        sim.step(5)
        outs.append(sim.get_psi())
        sim.close()
    assert np.array_equal(outs[0], outs[1])


@pytest.mark.parametrize("shape,mode", [((256, 256, 128), REAL), ((512, 256, 64), IMAG)])
def test_paced_and_unpaced_passes_agree_bitwise(gp, monkeypatch, shape, mode):
    """Fields larger than L2: the loaders of the streaming passes are paced to the slowest CTA of the launch
    (tma_pipe.cuh: pace_wait; DBEC_PACE=0 switches it off).  Pacing moves no arithmetic: bit-identical psi, and the
    lag word is back at zero after every launch."""
    w = grid3(*shape, mode)
    psi0 = random_psi(w, 23)
    outs = []
    for pace in (None, "0"):
        if pace is None:
            monkeypatch.delenv("DBEC_PACE", raising=False)
        else:
            monkeypatch.setenv("DBEC_PACE", pace)
        sim = gp.Dbec(gp.params_of(w))
        sim.set_psi(psi0)
        sim.step(4)
        outs.append(sim.get_psi())
        sim.close()
    assert np.array_equal(outs[0], outs[1])


def test_handles_on_concurrent_streams_do_not_disturb_each_other(gp):
    """Three handles on three streams advance at the same time: a paced 256 x 256 x 128 grid (its persistent kernels
    want every SM and wait for each other's lag word, which lives in each handle's own workspace), a 128^3 grid and a
    32^3 grid on its cluster.  Nothing may hang, and each result is bit-identical to the same handle run alone."""
    ws = [grid3(256, 256, 128, REAL), grid3(128, 128, 128, IMAG), grid3(32, 32, 32, REAL)]
    psis = [random_psi(w, 60 + i) for i, w in enumerate(ws)]
    alone = []
    for w, psi0 in zip(ws, psis):
        sim = gp.Dbec(gp.params_of(w))
        sim.set_psi(psi0)
        sim.step(6)
        alone.append(sim.get_psi())
        sim.close()
    sims = [gp.Dbec(gp.params_of(w)) for w in ws]
    for sim, psi0 in zip(sims, psis):
        sim.set_psi(psi0)
    for _ in range(3):                       # interleave the enqueues: the three streams run side by side
        for sim in sims:
            sim.step(2)
    for sim, ref in zip(sims, alone):
        assert np.array_equal(sim.get_psi(), ref)
        sim.close()


@pytest.mark.parametrize("w", [grid3(512, 256, 128, REAL), grid3(512, 256, 128, IMAG, d=(0.4, 0.3, 0.6)), grid3(256, 512, 256, REAL)], ids=wid)
def test_z_sweep_on_paired_row_tiles(gp, ob, w):
    """xy planes of 2 MiB or more: the z sweep works on tiles of 8 columns x 2 rows of y (k_cn_tma with TC = 16;
    C5 is the only BASELINE.json config that gets there, in imaginary time with 256 points along z)."""
    psi0 = random_psi(w, 17)
    p = ob.params_of(w)
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(psi0)
    sim.cn_sweep(2)
    assert relerr(sim.get_psi(), ob.cn_sweep(p, psi0, 2)) < PSI_TOL
    sim.set_psi(psi0)
    sim.step(1)
    o = ob.Oracle(p)
    o.set_psi(psi0)
    o.step(1)
    assert relerr(sim.get_psi(), o.get_psi()) < PSI_TOL
    sim.close()
    o.close()


CLUSTER_CASES = [grid3(32, 32, 32, IMAG), grid3(32, 32, 32, REAL), grid3(16, 16, 16, REAL), grid3(64, 16, 32, IMAG, d=(0.4, 0.3, 0.6)),
                 grid3(48, 20, 12, IMAG, d=(0.4, 0.3, 0.6)), grid3(50, 14, 6, REAL), grid3(12, 10, 6, IMAG), grid3(128, 32, 16, REAL),
                 grid3(16, 64, 64, IMAG), grid2(64, 32, REAL, dx=0.2, dy=0.3), grid2(256, 256, IMAG), grid2(96, 80, REAL, plane=1),
                 grid2(16, 1024, IMAG)]


@pytest.mark.parametrize("cs", ["1", "2", "8", "16"])
@pytest.mark.parametrize("w", CLUSTER_CASES, ids=wid)
def test_cluster_step_matches_oracle_and_multi_launch(gp, ob, w, cs, monkeypatch):
    """kernels_small.cu: the whole step in one launch by one thread-block cluster, several steps per
    launch, against the oracle and against the multi-launch path, for cluster sizes from 1 CTA (everything in one
    SM, ragged tiles) to 16; 2-D grids and run-time line lengths are forced onto it here."""
    psi0 = random_psi(w, 31)
    monkeypatch.setenv("DBEC_CLUSTER", cs)
    sim = gp.Dbec(gp.params_of(w))
    assert sim.pass_kernels() == {"sscn_step<cluster>": "k_small_step"}
    sim.set_psi(psi0)
    sim.step(3)
    got = sim.get_psi()
    obs = sim.observables()
    n0 = sim.launch_count()
    sim.step(5)
    assert sim.launch_count() - n0 == 1            # five steps, one launch
    sim.close()
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(psi0)
    o.step(3)
    assert relerr(got, o.get_psi()) < PSI_TOL
    b = o.observables()
    for k in b:
        if w.ndim == 2 and k == "rms_z":
            continue
        assert abs(obs[k] - b[k]) <= OBS_TOL * max(abs(b[k]), 1e-300), k
    o.close()
    monkeypatch.setenv("DBEC_CLUSTER", "0")
    ml = gp.Dbec(gp.params_of(w))
    assert "sscn_step<cluster>" not in ml.pass_kernels()
    ml.set_psi(psi0)
    ml.step(3)
    assert relerr(got, ml.get_psi()) < PSI_TOL
    ml.close()


@pytest.mark.parametrize("p2", ["1", "0"])
def test_cluster_step_batch_ramp_and_choice(gp, ob, monkeypatch, p2):
    """A batch on the cluster step (one cluster per member, per-member couplings, the NSTP ramp advancing inside a
    launch) and the automatic choice: small 3-D grids only, and only while every member gets a resident cluster.
    p2: with / without the variant compiled for power-of-two shapes (kernels_small_p2.cu)."""
    monkeypatch.delenv("DBEC_CLUSTER", raising=False)
    monkeypatch.setenv("DBEC_SMALL_P2", p2)
    w = grid3(32, 32, 32, IMAG, G=0.0, D=0.0)
    nb = 3
    psis = np.stack([random_psi(w, 50 + m) for m in range(nb)])
    sim = gp.Dbec(gp.params_of(w), nbatch=nb)
    assert sim.pass_kernels() == {"sscn_step<cluster>": "k_small_p2" if p2 == "1" else "k_small_step"}
    sim.set_psi(psis)
    sim.set_ramp(4, 0.0, 0.0, 40.0, 25.0)
    sim.step(6)                                       # the ramp ends inside the launch
    got = sim.get_psi()
    sim.close()
    for m in range(nb):
        o = ob.Oracle(ob.params_of(w))
        o.set_psi(psis[m])
        for k in range(1, 7):
            f = min(k, 4) / 4.0
            o.set_coupling(40.0 * f, 25.0 * f)
            o.step(1)
        assert relerr(got[m], o.get_psi()) < PSI_TOL, m
        o.close()
    # (k_small_p2 walks a batch through its resident clusters, k_small_step wants a cluster per member)
    for wl, nbatch, small in ((grid3(32, 32, 32, REAL), 1, True), (grid3(32, 32, 32, REAL), 200, p2 == "1"),
                              (grid2(128, 128, REAL), 1, False), (grid3(64, 64, 32, IMAG), 1, p2 == "1"),
                              (grid3(64, 64, 64, IMAG), 1, False)):
        h = gp.Dbec(gp.params_of(wl), nbatch=nbatch)
        assert ("sscn_step<cluster>" in h.pass_kernels()) == small, (wid(wl), nbatch)
        h.close()


@pytest.mark.parametrize("shape", P2_SHAPES)
@pytest.mark.parametrize("mode", [IMAG, REAL])
def test_power_of_two_cluster_step_matches_oracle_and_general_kernel(gp, ob, shape, mode, monkeypatch):
    """k_small_p2 on every shape it is compiled for: five steps in one launch against the oracle (imaginary time:
    the norm factor is carried from step to step inside the launch) and against k_small_step (beyond 64 Ki points:
    the multi-launch path) on the same input."""
    monkeypatch.delenv("DBEC_CLUSTER", raising=False)
    monkeypatch.delenv("DBEC_SMALL_P2", raising=False)
    w = grid3(*shape, mode, d=(0.4, 0.35, 0.5))
    psi0 = random_psi(w, 77) if mode == REAL else 1.3 * initial_psi(w)
    sim, o, got, ref = one_step_pair(gp, ob, w, psi0, steps=5)
    assert sim.pass_kernels() == {"sscn_step<cluster>": "k_small_p2"}
    assert relerr(got, ref) < 5 * PSI_TOL
    a, b = sim.observables(), o.observables()
    for k in b:
        assert abs(a[k] - b[k]) <= OBS_TOL * max(abs(b[k]), 1e-300), k
    sim.close()
    o.close()
    monkeypatch.setenv("DBEC_SMALL_P2", "0")
    gen = gp.Dbec(gp.params_of(w))
    if w.npoints <= 65536:
        assert gen.pass_kernels() == {"sscn_step<cluster>": "k_small_step"}
    else:                                      # beyond k_small_step's 64 Ki points: the multi-launch path
        assert "sscn_step<cluster>" not in gen.pass_kernels()
    gen.set_psi(psi0)
    gen.step(5)
    assert relerr(got, gen.get_psi()) < 5 * PSI_TOL
    gen.close()


@pytest.mark.parametrize("mode", [IMAG, REAL])
def test_async_host_copies_on_two_handles_match_the_synchronous_calls(gp, mode):
    """dbec_set_psi_async / dbec_get_psi_async / dbec_synchronize with pinned host buffers, two handles on two
    streams taking turns (the end-to-end leg of bench.py): every result is bitwise what dbec_set_psi, dbec_step,
    dbec_get_psi give on one handle."""
    import torch
    w = grid3(64, 32, 128, mode, d=(0.4, 0.3, 0.5))
    inputs = [random_psi(w, 90 + i) for i in range(5)]
    one = gp.Dbec(gp.params_of(w))
    want = []
    for psi in inputs:
        one.set_psi(psi)
        one.step(2)
        want.append(one.get_psi().copy())
    one.close()
    pair = [gp.Dbec(gp.params_of(w)) for _ in range(2)]
    h_in = [torch.from_numpy(psi.copy()).pin_memory() for psi in inputs]
    h_out = [torch.empty_like(h_in[0]).pin_memory() for _ in inputs]
    for i in range(len(inputs)):
        s = pair[i & 1]
        s.set_psi_async(h_in[i])
        s.step(2)
        s.get_psi_async(h_out[i])
    for s in pair:
        s.wait()
    for i in range(len(inputs)):
        assert np.array_equal(h_out[i].numpy(), want[i]), i
    for s in pair:
        s.close()


@pytest.mark.parametrize("n,cs,nb", [(32, 8, 1), (32, 8, 40), (32, 16, 21), (16, 4, 1), (16, 1, 1), (16, 1, 300), (16, 4, 75),
                                     (32, 4, 1), (32, 2, 1), (32, 2, 90), (32, 4, 50)])
@pytest.mark.parametrize("mode", [IMAG, REAL])
def test_power_of_two_cluster_step_cluster_sizes_and_batches(gp, ob, n, cs, nb, mode, monkeypatch):
    """k_small_p2 with fewer CTAs per cluster (DBEC_SMALL_P2_CS) and with more batch members than resident clusters
    (a cluster then works through several members one after the other): four steps in one launch against the
    oracle on the first, a middle and the last member."""
    monkeypatch.delenv("DBEC_CLUSTER", raising=False)
    monkeypatch.delenv("DBEC_SMALL_P2", raising=False)
    monkeypatch.setenv("DBEC_SMALL_P2_CS", str(cs))
    w = grid3(n, n, n, mode, d=(0.5, 0.45, 0.4))
    rng = np.random.default_rng(7)
    scale = 1.0 + 0.5 * rng.random(nb)
    base = random_psi(w, 31) if mode == REAL else initial_psi(w)
    psis = np.stack([scale[m] * base for m in range(nb)]) if nb > 1 else base
    sim = gp.Dbec(gp.params_of(w), nbatch=nb)
    assert sim.pass_kernels() == {"sscn_step<cluster>": "k_small_p2"}
    sim.set_psi(psis)
    sim.step(4)
    got = sim.get_psi()
    sim.close()
    for m in sorted({0, nb // 2, nb - 1}):
        o = ob.Oracle(ob.params_of(w))
        o.set_psi(psis[m] if nb > 1 else psis)
        o.step(4)
        assert relerr(got[m] if nb > 1 else got, o.get_psi()) < 5 * PSI_TOL, m
        o.close()


@pytest.mark.parametrize("shape,mode", [((256, 128, 256), REAL), ((128, 128, 128), IMAG), ((256, 256, 64), IMAG),
                                        ((512, 64, 64), REAL), ((512, 256, 32), IMAG)])
def test_persistent_kernels_are_bit_reproducible(gp, shape, mode):
    """The persistent loader / worker / storer kernels (kernels_tma.cu, kernels_xline.cu) hand stages over
    through mbarrier phase parities; a worker that ran a whole ring ahead once read a stage that was
    still in use (intermittently, only at full size).  Same input, repeated steps: bitwise equal."""
    w = grid3(*shape, mode, dx=0.1)
    psi0 = random_psi(w, seed=5)
    sim = gp.Dbec(gp.params_of(w))
    ref = None
    for rep in range(10):
        sim.set_psi(psi0)
        sim.step(2)
        got = sim.get_psi()
        if ref is None:
            ref = got.copy()
        else:
            assert np.array_equal(got, ref), f"repetition {rep} differs"
    sim.close()


def test_full_run_C1_observables(gp, ob):
    w = workload("C1")
    psi0 = initial_psi(w)
    sim, o, got, ref = one_step_pair(gp, ob, w, psi0, steps=w.steps)
    assert relerr(got, ref) < 1e-10
    a, b = sim.observables(), o.observables()
    for k in ("norm", "mu", "energy", "rms_x", "rms_y", "rms_z", "rms_r", "density0"):
        assert abs(a[k] - b[k]) <= OBS_TOL * abs(b[k]), k
    sim.close()
    o.close()


def test_real_time_norm_conserved_on_gpu(gp):
    w = workload("C2")
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(initial_psi(w))
    sim.set_coupling(w.G_run, w.D_run)
    sim.step(100)
    assert abs(sim.observables()["norm"] - 1.0) < 1e-12
    sim.close()


# ------------------------------------------------------------------ f2: line lengths that are not powers of two
GEN3 = [(96, 80, 48), (48, 20, 12), (50, 14, 6), (1024, 8, 4), (12, 1024, 4), (6, 10, 600), (256, 96, 40), (80, 128, 256),
        (16, 24, 32)]
GEN2 = [(96, 80), (1000, 12), (50, 70), (512, 48), (48, 512), (1024, 1024)]


def gen_workloads():
    out = []
    for mode in (IMAG, REAL):
        for s in GEN3:
            out.append(grid3(*s, mode, d=(0.4, 0.3, 0.6)))
        for s in GEN2:
            out.append(grid2(*s, mode, dx=0.2, dy=0.25, plane=(s[0] // 2) % 2))
    return out


@pytest.mark.parametrize("w", gen_workloads(), ids=wid)
def test_non_power_of_two_lengths(gp, ob, w):
    """Every part and one full step on grids whose lines run in the run-time-length kernels (kernels_gen.cu), mixed
    with axes the register-resident / persistent kernels serve."""
    psi0 = random_psi(w, 9)
    p = ob.params_of(w)
    sim = gp.Dbec(gp.params_of(w))
    for axis in range(w.ndim):
        sim.set_psi(psi0)
        sim.cn_sweep(axis)
        assert relerr(sim.get_psi(), ob.cn_sweep(p, psi0, axis)) < PSI_TOL, f"cn axis {axis}"
    sim.set_psi(psi0)
    phi = ob.phi_dd(p, np.abs(psi0) ** 2)
    assert relerr(sim.phi_dd().cpu().numpy(), phi) < PSI_TOL
    sim.nonlinear()
    assert relerr(sim.get_psi(), ob.nonlinear(p, psi0, phi)) < PSI_TOL
    sim.set_psi(psi0)
    sim.step(2)
    o = ob.Oracle(p)
    o.set_psi(psi0)
    o.step(2)
    assert relerr(sim.get_psi(), o.get_psi()) < PSI_TOL
    a, b = sim.observables(), o.observables()
    for k in b:
        if w.ndim == 2 and k == "rms_z":
            continue
        assert abs(a[k] - b[k]) <= OBS_TOL * max(abs(b[k]), 1e-300), k
    sim.close()
    o.close()


def test_non_power_of_two_batch_and_ramp(gp, ob):
    w = grid3(48, 20, 12, IMAG, d=(0.4, 0.3, 0.6))
    nb = 3
    psis = np.stack([initial_psi(w, noise=1e-3 * (m + 1)) for m in range(nb)])
    sim = gp.Dbec(gp.params_of(w), nbatch=nb)
    sim.set_psi(psis)
    sim.set_ramp(3, 0.0, 0.0, w.G, w.D)
    sim.step(4)
    got = sim.get_psi()
    for m in range(nb):
        o = ob.Oracle(ob.params_of(w))
        o.set_psi(psis[m])
        o.set_ramp(3, 0.0, 0.0, w.G, w.D)
        o.step(4)
        assert relerr(got[m], o.get_psi()) < PSI_TOL, m
        o.close()
    sim.close()


def test_errors_and_edge_cases(gp):
    import ctypes as C
    L = gp.lib()
    p = gp.params(3, 44, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0)
    n = C.c_size_t()
    assert L.dbec_workspace_bytes(C.byref(p), C.byref(n)) == gp.DBEC_ESIZE
    p = gp.params(3, 32, 32, 32, .5, .5, .5, -1.0, 1, 1, .5, 1, 1, 0)
    assert L.dbec_workspace_bytes(C.byref(p), C.byref(n)) == gp.DBEC_EINVAL
    p = gp.params(3, 32, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0)
    h = C.c_void_p()
    assert L.dbec_create(C.byref(p), None, 0, None, C.byref(h)) == gp.DBEC_EWORKSPACE
    assert L.dbec_step(None, 1) == gp.DBEC_EINVAL
    sim = gp.Dbec(p)
    assert L.dbec_step(sim._h, -1) == gp.DBEC_EINVAL
    sim.step(0)                      # zero steps: nothing happens
    assert np.all(sim.get_psi() == 0)
    assert sim.launch_count() >= 1
    sim.close()


# ------------------------------------------------------------------ f3: run protocol (readings S26, S27)
@pytest.mark.parametrize("w", [grid3(32, 32, 32, IMAG, G=0.0, D=0.0), grid3(128, 16, 32, REAL, G=0.0, D=0.0),
                               grid2(256, 128, REAL, G=0.0, D=0.0), grid2(32, 64, IMAG, G=0.0, D=0.0)], ids=wid)
def test_nstp_ramp_matches_oracle(gp, ob, w):
    """dbec_set_ramp: the schedule lives in device scalars that the first kernel of every step advances, so the
    replayed CUDA graph sees it; observables in between must not advance it."""
    psi0 = random_psi(w, 9) if w.time_mode == REAL else initial_psi(w)
    sim = gp.Dbec(gp.params_of(w))
    o = ob.Oracle(ob.params_of(w))
    sim.set_psi(psi0)
    o.set_psi(psi0)
    sim.set_ramp(5, 1.0, 0.5, 30.0, 18.0)
    o.set_ramp(5, 1.0, 0.5, 30.0, 18.0)
    for n in (2, 1, 4):                                # 7 steps: the ramp ends inside the last call
        sim.step(n)
        o.step(n)
        a, b = sim.observables(), o.observables()      # uses the CURRENT ramp value of G and D in mu / E
        for k in ("norm", "mu", "energy", "rms_x", "rms_y"):
            assert abs(a[k] - b[k]) <= OBS_TOL * abs(b[k]), (n, k)
        assert relerr(sim.get_psi(), o.get_psi()) < PSI_TOL
    for x in (sim, o):                                 # an explicit value ends a running ramp
        x.set_ramp(3, 0.0, 0.0, 9.0, 6.0)
        x.step(1)
        x.set_coupling(7.0, 3.0)
        x.step(2)
    assert relerr(sim.get_psi(), o.get_psi()) < PSI_TOL
    sim.close()
    o.close()


def test_imag_to_real_handoff_on_device(gp, ob):
    """The paper's NSTP = 0 restart: a real-time run starts from the state an
    imaginary-time run produced.  Here the state goes from one handle to the other as a DEVICE buffer."""
    import torch
    w = grid3(32, 32, 64, IMAG, G=20.0, D=10.0)
    from dataclasses import replace
    wr = replace(w, time_mode=REAL, dt=0.5 * w.dx ** 2)
    psi0 = initial_psi(w)
    a = gp.Dbec(gp.params_of(w))
    b = gp.Dbec(gp.params_of(wr))
    a.set_psi(psi0)
    a.step(20)
    buf = torch.empty(w.shape, dtype=torch.complex128, device="cuda")
    a.get_psi(buf)                                     # applies the deferred norm factor
    b.set_psi(buf)
    b.set_ramp(0, 0.0, 0.0, 25.0, 12.0)                # NSTP = 0: end values at once
    b.step(5)
    got = b.get_psi()
    oa = ob.Oracle(ob.params_of(w))
    oa.set_psi(psi0)
    oa.step(20)
    orr = ob.Oracle(ob.params_of(wr))
    orr.set_psi(oa.get_psi())
    orr.set_ramp(0, 0.0, 0.0, 25.0, 12.0)
    orr.step(5)
    assert relerr(got, orr.get_psi()) < 1e-11           # 25 steps of round-off
    assert abs(b.observables()["norm"] - 1.0) < 1e-12
    for s in (a, b):
        s.close()


@pytest.mark.parametrize("w", [grid3(32, 16, 64, IMAG, d=(0.4, 0.3, 0.6)), grid3(128, 128, 128, REAL),
                               grid2(64, 32, REAL, dy=0.3), grid2(512, 256, IMAG)], ids=wid)
def test_integrated_densities_match_oracle(gp, ob, w):
    psi0 = random_psi(w, 12)
    sim = gp.Dbec(gp.params_of(w))
    o = ob.Oracle(ob.params_of(w))
    sim.set_psi(1.3 * psi0)
    o.set_psi(1.3 * psi0)
    if w.time_mode == IMAG:                            # leaves a deferred norm factor in the handle
        sim.step(1)
        o.step(1)
    for ax in range(w.ndim):
        assert relerr(sim.density_1d(ax), o.density_1d(ax)) < PSI_TOL, ax
    if w.ndim == 3:
        for ax in range(3):
            assert relerr(sim.density_2d(ax), o.density_2d(ax)) < PSI_TOL, ax
    else:
        import ctypes as C
        buf = np.empty(8)
        assert gp.lib().dbec_density_2d(sim._h, 0, 0, C.c_void_p(buf.ctypes.data), 0) == gp.DBEC_EINVAL
    # the observables still work afterwards (the densities borrow their scratch buffer)
    assert abs(sim.observables()["mu"] - o.observables()["mu"]) <= OBS_TOL * abs(o.observables()["mu"])
    sim.close()
    o.close()


# ------------------------------------------------------------------ f4: batched handles
BATCH_CASES = [(grid3(32, 32, 32, IMAG), 5), (grid3(32, 32, 32, REAL), 3), (grid3(16, 64, 32, IMAG), 4),
               (grid3(128, 16, 16, REAL), 3), (grid3(128, 32, 128, IMAG), 2), (grid2(512, 512, REAL), 3),
               (grid2(256, 128, IMAG), 4), (grid2(32, 64, IMAG), 7), (grid2(128, 16, REAL, plane=1), 3)]


@pytest.mark.parametrize("w,nb", BATCH_CASES, ids=[f"{wid(w)}-x{nb}" for w, nb in BATCH_CASES])
def test_batch_members_match_single_oracle_runs(gp, ob, w, nb):
    """dbec_create_batch: nb independent members (different psi, different G and D) advance in the same
    launches; each must match its own oracle run, observables included."""
    psis = np.stack([(1.0 + 0.1 * m) * (random_psi(w, 30 + m) if w.time_mode == REAL else initial_psi(w, noise=1e-3 * (m + 1)))
                     for m in range(nb)])
    Gs = np.array([w.G * (1 + 0.2 * m) for m in range(nb)])
    Ds = np.array([w.D * (1 - 0.1 * m) for m in range(nb)])
    sim = gp.Dbec(gp.params_of(w), nbatch=nb)
    assert sim.shape == (nb,) + w.shape
    sim.set_psi(psis)
    sim.set_coupling(Gs, Ds)
    sim.step(3)
    got = sim.get_psi()
    obs = sim.observables()
    assert len(obs) == nb
    for m in range(nb):
        o = ob.Oracle(ob.params_of(w, G=Gs[m], D=Ds[m]))
        o.set_psi(psis[m])
        o.step(3)
        assert relerr(got[m], o.get_psi()) < PSI_TOL, m
        b = o.observables()
        for k in b:
            if w.ndim == 2 and k == "rms_z":
                continue
            assert abs(obs[m][k] - b[k]) <= OBS_TOL * max(abs(b[k]), 1e-300), (m, k)
        if m == nb - 1:
            assert relerr(sim.density_1d(0, member=m), o.density_1d(0)) < PSI_TOL
        o.close()
    # the single-part entry points act on every member
    sim.set_psi(psis)
    sim.cn_sweep(1)
    sim.normalize()
    got = sim.get_psi()
    for m in (0, nb - 1):
        p = ob.params_of(w)
        ref = ob.normalize(p, ob.cn_sweep(p, psis[m], 1))
        assert relerr(got[m], ref) < PSI_TOL, m
    import ctypes as C
    one = gp.DbecObs()
    assert gp.lib().dbec_observables(sim._h, C.byref(one)) == gp.DBEC_EINVAL
    sim.close()


def test_batch_is_bitwise_the_single_handle(gp):
    """Member m of a batch goes through the same arithmetic as a handle of its own."""
    for w, nb in ((grid3(32, 32, 32, IMAG), 3), (grid2(256, 128, REAL), 2)):
        psis = np.stack([random_psi(w, 40 + m) for m in range(nb)])
        sim = gp.Dbec(gp.params_of(w), nbatch=nb)
        sim.set_psi(psis)
        sim.step(4)
        got = sim.get_psi()
        sim.close()
        for m in range(nb):
            one = gp.Dbec(gp.params_of(w))
            one.set_psi(psis[m])
            one.step(4)
            assert np.array_equal(one.get_psi(), got[m]), (wid(w), m)
            one.close()


def test_workspace_guard_bands_stay_intact(gp):
    """compute-sanitizer is not available on this pool: instead, every persistent / one-tile-per-block kernel
    runs on a workspace with 1 MiB guard bands on both sides (and between nothing else the caller owns); a
    bulk or TMA store that leaves the workspace would land in them."""
    import ctypes as C
    import torch
    L = gp.lib()
    shapes = [grid3(32, 32, 32, IMAG), grid3(128, 128, 128, REAL), grid3(256, 16, 16, IMAG), grid3(16, 256, 32, REAL),
              grid3(32, 16, 512, IMAG), grid2(512, 512, REAL), grid2(16, 16, IMAG), grid2(128, 256, IMAG, plane=1)]
    for w in shapes:
        for nb in (1, 3):
            p = gp.params_of(w)
            n = C.c_size_t()
            assert L.dbec_workspace_bytes_batch(C.byref(p), nb, C.byref(n)) == 0
            G = 1 << 20
            buf = torch.full((n.value + 2 * G,), 0xA5, dtype=torch.uint8, device="cuda")
            st = torch.cuda.Stream()
            torch.cuda.synchronize()
            h = C.c_void_p()
            assert L.dbec_create_batch(C.byref(p), nb, C.c_void_p(buf.data_ptr() + G), n.value, C.c_void_p(st.cuda_stream), C.byref(h)) == 0
            psi = np.stack([random_psi(w, 3 + m) for m in range(nb)])
            assert L.dbec_set_psi(h, C.c_void_p(psi.ctypes.data), 0) == 0
            assert L.dbec_step(h, 3) == 0
            obs = (gp.DbecObs * nb)()
            assert L.dbec_observables_batch(h, obs) == 0
            out = np.empty_like(psi)
            assert L.dbec_get_psi(h, C.c_void_p(out.ctypes.data), 0) == 0
            assert L.dbec_destroy(h) == 0
            torch.cuda.synchronize()
            assert bool((buf[:G] == 0xA5).all()) and bool((buf[-G:] == 0xA5).all()), (wid(w), nb)
            assert np.all(np.isfinite(out.view(np.float64)))


GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.mark.parametrize("key", ["C1", "C2", "C3", "C4", "C5", "X0", "X1", "X2"])
def test_full_run_observables_against_oracle_golden(gp, key):
    """BASELINE.json: mu, energy, rms after the full run within 1e-9 relative.  The expected values were
    written by tests/golden/make_golden.py, which calls only oracle/ (full oracle runs of C3-C5 take
    tens of minutes, too long for this suite)."""
    path = os.path.join(GOLDEN, f"{key}.json")
    if not os.path.exists(path):
        pytest.skip(f"no oracle golden file for {key} yet")
    with open(path) as f:
        gold = json.load(f)
    w = workload(key)
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(initial_psi(w))
    if (w.G_run, w.D_run) != (w.G, w.D):
        sim.set_coupling(w.G_run, w.D_run)
    done = 0
    for row in gold["observables"]:
        sim.step(row["step"] - done)
        done = row["step"]
        a = sim.observables()
        for k in ("norm", "mu", "energy", "rms_x", "rms_y", "rms_z", "rms_r", "density0"):
            if w.ndim == 2 and k == "rms_z":
                continue
            assert abs(a[k] - row[k]) <= OBS_TOL * abs(row[k]), (key, row["step"], k, a[k], row[k])
    assert done == w.steps
    sim.close()


@pytest.mark.gpu
def test_fp64_pipe_probe(tmp_path):
    """Builds and runs tests/fp64_probe.cu: dependent-DFMA latency and DFMA throughput per SM, the two numbers
    DESIGN.md section 6 sets beside the HBM roofline (profiles/r2_fp64_probe.md keeps one run's line)."""
    import json
    import shutil
    import subprocess
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("no nvcc on this box")
    exe = str(tmp_path / "fp64_probe")
    src = os.path.join(os.path.dirname(__file__), "fp64_probe.cu")
    subprocess.run([nvcc, "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe, src], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stdout + r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    print("fp64_probe", json.dumps(line))
    assert line["cuda_error"] == 0
    assert 4.0 <= line["dependent_dfma_latency_cycles"] <= 16.0
    assert 16.0 <= line["dfma_per_clk_per_sm"] <= 130.0
