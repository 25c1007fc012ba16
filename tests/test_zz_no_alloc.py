"""dbec_norm_noalloc (include/dbec.h): the norm integral through the entry point that allocates nothing, against
the existing path (dbec_observables on a handle holding the same field) and against the definition
dV * sum |psi|^2 in numpy fp64.  Tolerance: the 1e-12 relative bar of tests/test_gpu_parity.py.

Collected last on purpose (the file name): the suite runs with pytest -x.
"""
import numpy as np
import pytest

from paper_1601_04640_b200.inputs import IMAG, Workload, random_psi

pytestmark = pytest.mark.gpu

TOL = 1e-12


def grid3(nx, ny, nz, dx=0.4):
    return Workload("na3", 3, nx, ny, nz, dx, dx, dx, 0.1 * dx ** 2, 1.0, 1.2, 0.7, 30.0, 20.0, 30.0, 20.0, IMAG, 1, 31, 1)


@pytest.fixture(scope="module")
def gp():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1601_04640_b200 import dbec
    dbec.lib()
    return dbec


def existing_norm(gp, w, psi):
    sim = gp.Dbec(gp.params_of(w))
    sim.set_psi(psi)
    n = sim.observables()["norm"]
    sim.close()
    return n


def test_norm_noalloc_matches_existing_path_on_calls_in_a_row(gp):
    import torch
    # 17280 points = 4 blocks and a ragged tail; 524288 points = 128 blocks; 4096 points = exactly one block
    cases = [(grid3(48, 20, 18), 3, 1.7), (grid3(128, 64, 64), 4, 0.6), (grid3(16, 16, 16), 5, 2.5)]
    fields = []
    for w, seed, scale in cases:
        psi = scale * random_psi(w, seed)                   # not normalised: the answer is scale^2, not 1
        fields.append((w, psi, existing_norm(gp, w, psi), float(np.sum(np.abs(psi) ** 2)) * w.cell_volume))
    out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    dev = [torch.from_numpy(psi).to("cuda:0").contiguous() for _, psi, _, _ in fields]
    torch.cuda.synchronize()
    # big, small, big again, one block: a later call finds the earlier calls' partial sums in the shared scratch
    order = [1, 0, 1, 2, 0, 0]
    for n, k in enumerate(order):
        w, psi, ref_path, ref_def = fields[k]
        out.fill_(-1.0)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info(0)[0]
        gp.norm_noalloc(dev[k].reshape(-1), w.cell_volume, out=out)
        torch.cuda.synchronize()
        free1 = torch.cuda.mem_get_info(0)[0]
        got = float(out.item())
        assert abs(got - ref_path) <= TOL * abs(ref_path), (n, k, got, ref_path)
        assert abs(got - ref_def) <= TOL * abs(ref_def), (n, k, got, ref_def)
        if n > 0:       # (the first call may load the module lazily)
            assert free1 == free0, f"call {n} changed the device's free memory by {free0 - free1} bytes"
    # bit-identical from call to call: fixed summation order, whatever the scratch held before
    w, psi, _, _ = fields[1]
    vals = []
    for _ in range(3):
        gp.norm_noalloc(dev[1].reshape(-1), w.cell_volume, out=out)
        vals.append(float(out.item()))
    assert vals[0] == vals[1] == vals[2]


def test_norm_noalloc_on_a_side_stream(gp):
    import torch
    w = grid3(64, 32, 32)
    psi = 1.3 * random_psi(w, 9)
    ref = existing_norm(gp, w, psi)
    d = torch.from_numpy(psi).to("cuda:0").reshape(-1)
    out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    torch.cuda.synchronize()
    st = torch.cuda.Stream(device="cuda:0")
    for _ in range(2):
        gp.norm_noalloc(d, w.cell_volume, out=out, stream=st)
        st.synchronize()
        assert abs(float(out.item()) - ref) <= TOL * abs(ref)


def test_norm_noalloc_rejects_bad_arguments(gp):
    import torch
    L = gp.lib()
    d = torch.zeros(4096, dtype=torch.complex128, device="cuda:0")
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda:0")
    torch.cuda.synchronize()
    st = torch.cuda.current_stream().cuda_stream
    too_many = gp.NOALLOC_MAX_POINTS + 1
    rc = L.dbec_norm_noalloc(d.data_ptr(), too_many, 1.0, out.data_ptr(), st)      # refused before anything is read
    assert rc == -6
    assert b"DBEC_NOALLOC_MAX_POINTS" in L.dbec_strerror(rc)
    assert L.dbec_norm_noalloc(None, 4096, 1.0, out.data_ptr(), st) == -1
    assert L.dbec_norm_noalloc(d.data_ptr(), 4096, 1.0, None, st) == -1
    assert L.dbec_norm_noalloc(d.data_ptr(), 0, 1.0, out.data_ptr(), st) == -1
    assert L.dbec_norm_noalloc(d.data_ptr(), 4096, 0.0, out.data_ptr(), st) == -1
    torch.cuda.synchronize()
    assert float(out.item()) == 7.0                                                 # no refused call wrote anything
    # the largest size the scratch serves is accepted (2 GiB of psi: only on a device with the room)
    if torch.cuda.mem_get_info(0)[0] > 3 * (1 << 30):
        big = torch.zeros(gp.NOALLOC_MAX_POINTS, dtype=torch.complex128, device="cuda:0")
        big[::4097] = 1.0 + 1.0j
        cnt = (gp.NOALLOC_MAX_POINTS + 4096) // 4097
        gp.norm_noalloc(big, 0.5, out=out)
        torch.cuda.synchronize()
        assert float(out.item()) == 0.5 * 2.0 * cnt
        del big
