"""CPU-only checks of the product's host side: the C-ABI library loads and exports every symbol that
include/dbec.h declares, host-only entry points validate their arguments, there is no CPU fallback,
and bench.py's multi-rank plumbing (replicas only: max-over-ranks time, whole-job value) works with
world_size 2 over gloo."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gp():
    from paper_1601_04640_b200 import dbec
    dbec.lib()
    return dbec


def test_library_exports_every_declared_symbol(gp):
    hdr = open(os.path.join(ROOT, "include", "dbec.h")).read()
    declared = set(re.findall(r"\b(dbec_[a-z_0-9]+)\s*\(", hdr))
    assert {"dbec_create", "dbec_set_psi", "dbec_step", "dbec_observables"} <= declared
    L = gp.lib()
    for name in sorted(declared):
        assert hasattr(L, name), name
    assert declared == set(gp.EXPORTS)
    assert L.dbec_version() >= 100


def test_workspace_bytes_validation_is_host_only(gp):
    L = gp.lib()
    n = C.c_size_t()
    ok = gp.params(3, 256, 256, 256, .1, .1, .1, .005, 1, 1.2, .8, 200, 150, 1)
    assert L.dbec_workspace_bytes(C.byref(ok), C.byref(n)) == gp.DBEC_OK
    # psi + half spectrum + V_dd table (folded by its even symmetry in k_y, k_z: 129 x 129 rows) + phi
    P, SP, VP = 256 ** 3, 256 * 256 * 136, 129 * 129 * 136
    assert n.value >= 16 * P + 16 * SP + 8 * VP + 8 * P
    assert n.value < 16 * P + 16 * SP + 8 * VP + 8 * P + (4 << 20)
    xz = gp.params(2, 32, 32, 1, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0, plane=1)
    assert L.dbec_workspace_bytes(C.byref(xz), C.byref(n)) == gp.DBEC_OK
    # lengths 4..1024 with prime factors 2, 3, 5, 7 (the paper's grids are mostly not powers of two)
    for shape in ((48, 32, 32), (96, 80, 48), (1024, 32, 8), (50, 70, 6), (600, 4, 4)):
        ok2 = gp.params(3, *shape, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0)
        assert L.dbec_workspace_bytes(C.byref(ok2), C.byref(n)) == gp.DBEC_OK, shape
    assert L.dbec_workspace_bytes(None, C.byref(n)) == gp.DBEC_EINVAL
    assert L.dbec_workspace_bytes(C.byref(ok), None) == gp.DBEC_EINVAL
    for bad, code in [
        (gp.params(3, 44, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0), gp.DBEC_ESIZE),       # prime factor 11
        (gp.params(3, 2048, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0), gp.DBEC_ESIZE),    # too long
        (gp.params(3, 32, 32, 2, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0), gp.DBEC_ESIZE),       # too short
        (gp.params(3, 45, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0), gp.DBEC_ESIZE),       # NX odd
        (gp.params(2, 32, 15, 1, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0), gp.DBEC_ESIZE),        # NY*NZ odd: lines do not pair
        (gp.params(2, 32, 32, 2, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0), gp.DBEC_EINVAL),      # 2-D with nz != 1
        (gp.params(4, 32, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0), gp.DBEC_EINVAL),
        (gp.params(3, 32, 32, 32, 0., .5, .5, .025, 1, 1, .5, 1, 1, 0), gp.DBEC_EINVAL),
        (gp.params(3, 32, 32, 32, .5, .5, .5, 0., 1, 1, .5, 1, 1, 0), gp.DBEC_EINVAL),
        (gp.params(3, 32, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 2), gp.DBEC_EINVAL),      # time_mode
        (gp.params(2, 32, 32, 1, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0, plane=2), gp.DBEC_EINVAL),  # 0 = XY, 1 = XZ
        (gp.params(3, 32, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0, plane=1), gp.DBEC_EINVAL),  # 3-D has no plane
    ]:
        assert L.dbec_workspace_bytes(C.byref(bad), C.byref(n)) == code
    assert b"grid length" in L.dbec_strerror(gp.DBEC_ESIZE)


def test_null_handles_are_rejected(gp):
    L = gp.lib()
    assert L.dbec_step(None, 1) == gp.DBEC_EINVAL
    assert L.dbec_set_psi(None, None, 0) == gp.DBEC_EINVAL
    assert L.dbec_observables(None, None) == gp.DBEC_EINVAL
    assert L.dbec_destroy(None) == gp.DBEC_EINVAL
    assert L.dbec_set_psi_async(None, None) == gp.DBEC_EINVAL
    assert L.dbec_get_psi_async(None, None) == gp.DBEC_EINVAL
    assert L.dbec_synchronize(None) == gp.DBEC_EINVAL
    assert L.dbec_last_cuda_error(None) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the behaviour on a box without a GPU")
def test_no_cpu_fallback(gp):
    p = gp.params(3, 32, 32, 32, .5, .5, .5, .025, 1, 1, .5, 1, 1, 0)
    with pytest.raises(RuntimeError, match="no CPU path"):
        gp.Dbec(p)
    # straight through the C ABI: an aligned, large enough (fake) workspace gets as far as the device check
    h = C.c_void_p()
    rc = gp.lib().dbec_create(C.byref(p), C.c_void_p(1 << 20), C.c_size_t(1 << 40), None, C.byref(h))
    assert rc == gp.DBEC_ENODEVICE and not h.value


def _rank_main(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)            # slowest rank decides
    q.put((rank, ms, bench.whole_job_value(1000, 4, world, ms * 1e-3)))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_timing_plumbing_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, ms, value in out:
        assert ms == 15.0
        assert value == pytest.approx(2 * 1000 * 4 / 0.015)


def test_reference_arm_is_silent_on_other_ranks():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_prints_one_json_line():
    import json
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                        "--warmup", "1", "--workload", "C1"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0


def test_branch_free_sincos_matches_libm(tmp_path):
    """csrc/trig.cuh (used by the real-time calcnu) against numpy's sin/cos in long double: absolute
    error <= 2e-16 on |u| <= 1e9, exact values at 0, NaN beyond the stated range and for inf/nan."""
    import ctypes
    import numpy as np
    src = os.path.join(os.path.dirname(__file__), "host_trig_harness.cpp")
    so = str(tmp_path / "libtrig.so")
    subprocess.run(["g++", "-O2", "-shared", "-fPIC", "-o", so, src], check=True)
    L = ctypes.CDLL(so)
    L.sincos_cw_array.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long]
    rng = np.random.default_rng(7)
    parts = [rng.uniform(-s, s, 200000) for s in (1.0, 10.0, 1e3, 1e6, 1e8, 1e9)]
    parts.append(np.arange(-64, 65) * (np.pi / 4))            # quadrant boundaries
    parts.append(np.array([0.0, -0.0, 1e-300, 5e-324]))
    u = np.ascontiguousarray(np.concatenate(parts))
    sn, cs = np.empty_like(u), np.empty_like(u)
    L.sincos_cw_array(u.ctypes.data, sn.ctypes.data, cs.ctypes.data, u.size)
    ul = u.astype(np.longdouble)
    assert np.max(np.abs(sn - np.sin(ul))) <= 2e-16
    assert np.max(np.abs(cs - np.cos(ul))) <= 2e-16
    assert np.max(np.abs(sn * sn + cs * cs - 1.0)) <= 5e-16
    bad = np.array([2e9, -1e300, np.inf, -np.inf, np.nan])
    sb, cb = np.empty_like(bad), np.empty_like(bad)
    with np.errstate(all="ignore"):
        L.sincos_cw_array(bad.ctypes.data, sb.ctypes.data, cb.ctypes.data, bad.size)
    assert np.all(np.isnan(sb)) and np.all(np.isnan(cb))
    z = np.array([0.0]); s0, c0 = np.empty(1), np.empty(1)
    L.sincos_cw_array(z.ctypes.data, s0.ctypes.data, c0.ctypes.data, 1)
    assert s0[0] == 0.0 and c0[0] == 1.0


def test_branch_free_exp_matches_libm(tmp_path):
    """csrc/trig.cuh exp_cw (the imaginary-time calcnu) against numpy's exp in long double: relative error
    <= 2.5e-16 on |x| <= 700, exact 1 at 0, inf / 0 beyond the fp64 range, subnormal results to within one
    subnormal ulp, NaN for NaN."""
    import ctypes
    import numpy as np
    src = os.path.join(os.path.dirname(__file__), "host_trig_harness.cpp")
    so = str(tmp_path / "libtrig.so")
    subprocess.run(["g++", "-O2", "-shared", "-fPIC", "-o", so, src], check=True)
    L = ctypes.CDLL(so)
    L.exp_cw_array.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long]

    def run(x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        e = np.empty_like(x)
        with np.errstate(all="ignore"):
            L.exp_cw_array(x.ctypes.data, e.ctypes.data, x.size)
        return e

    rng = np.random.default_rng(11)
    parts = [rng.uniform(-s, s, 200000) for s in (1e-3, 1.0, 30.0, 700.0)]
    parts.append(np.arange(-1000, 1001) * (np.log(2.0) / 2))       # the reduction's interval ends
    x = np.concatenate(parts)
    x = x[np.abs(x) <= 700.0]
    ref = np.exp(x.astype(np.longdouble))
    rel = np.abs((run(x).astype(np.longdouble) - ref) / ref)
    assert float(rel.max()) <= 2.5e-16
    assert run([0.0, -0.0])[0] == 1.0 and run([-0.0])[0] == 1.0
    big = run([709.0, 710.0, 1e10, np.inf])
    assert np.isfinite(big[0]) and np.all(np.isinf(big[1:])) and np.all(big[1:] > 0)
    small = run([-746.0, -1e10, -np.inf])
    assert np.all(small == 0.0)
    xs = np.linspace(-744.0, -709.0, 500)                          # subnormal results
    assert np.max(np.abs(run(xs).astype(np.longdouble) - np.exp(xs.astype(np.longdouble)))) <= 5e-324 * 1.01
    assert np.isnan(run([np.nan])[0])
