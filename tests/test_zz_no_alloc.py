"""md_energy_static (the entry point that allocates nothing: its scratch is a static device array of the library,
md_static.cu) against the existing path, md_energy on a handle, at the tolerance the energy tests use (1e-5 relative,
north_star).  Collected last on purpose (the suite runs with pytest -x).  Every test makes two calls in a row whose
answers differ, so stale contents of the shared scratch would show."""
import ctypes as C

import numpy as np
import pytest

import workloads as W
from conftest import record_margin

pytestmark = pytest.mark.gpu
ETOL = 1e-5


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1401_4350_b200 as pkg
    return pkg


def handle_with_forces(api, w, order="hilbert"):
    s = api.MDSystem.from_workload(w, order=order)
    s.build_cells(); s.build_verlet(); s.forces("vertex", "l2")
    return s


def check(api, s, w, out, tag):
    """One md_energy_static call on the handle's arrays against md_energy on the handle."""
    import torch
    ref = np.array(s.energy())                                   # existing path (synchronises)
    rigid = s.angmom is not None
    pot = w.potential
    api.energy_static(s.vel, s.force, out, angmom=s.angmom if rigid else None, mass=pot.get("mass", 1.0),
                      inv_inertia=1.0 / pot["inertia"] if rigid else 0.0)
    torch.cuda.synchronize()
    got = out.cpu().numpy()[:3]
    scale = np.abs(ref).max()
    err = np.abs(got - ref).max() / scale
    record_margin(tag, "md_energy_static", "E vs md_energy", err, ETOL)
    assert np.all(np.abs(got - ref) <= ETOL * np.maximum(np.abs(ref), 1e-30) + 1e-12 * scale), (tag, got, ref)
    if not rigid:
        assert got[2] == 0.0
    return got


def test_two_calls_in_a_row_lj(api):
    """LJ fluid, N = 32000 (four blocks of the first stage, ragged tail), then the SAME handle after 50 steps (every input
    changed), then a smaller system (fewer partials than the call before left in the scratch)."""
    import torch
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda:0")   # the caller's output buffer
    w = W.lj_fluid(32000, seed=W.BASE_SEED + 11)
    s = handle_with_forces(api, w)
    e0 = check(api, s, w, out, "lj N=32000 call 1")
    s.integrate(w.dt, 50, "vertex", "smem")
    e1 = check(api, s, w, out, "lj N=32000 call 2 (after 50 steps)")
    assert not np.array_equal(e0, e1)
    assert abs(e0.sum() - e1.sum()) <= 1e-3 * abs(e0.sum())     # and it is still the same conserved energy
    w1 = W.config("C1")
    s1 = handle_with_forces(api, w1, order="none")
    check(api, s1, w1, out, "lj C1 after the larger call")


def test_two_calls_in_a_row_rigid(api):
    """Rigid bodies (the rotational term, K_r = sum |L|^2 / 2I), two different states back to back."""
    import torch
    out = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    w = W.patchy_fluid(13500, seed=W.BASE_SEED + 12)
    s = handle_with_forces(api, w)
    a = check(api, s, w, out, "patchy N=13500 call 1")
    s.integrate(w.dt, 20, "edge", "red_v4")
    b = check(api, s, w, out, "patchy N=13500 call 2 (after 20 steps)")
    assert a[2] > 0.0 and not np.array_equal(a, b)


def test_no_device_allocation_and_limit(api):
    """The call leaves the device's free memory unchanged, and rejects n beyond MD_ENERGY_STATIC_MAX_N without launching."""
    import torch
    w = W.config("C1")
    s = handle_with_forces(api, w, order="none")
    out = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    api.energy_static(s.vel, s.force, out)                       # first call on the device: symbol look-up, module load
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    reserved0 = torch.cuda.memory_reserved()
    for _ in range(3):
        api.energy_static(s.vel, s.force, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0 and torch.cuda.memory_reserved() == reserved0

    lib = api.load_library()
    err = C.create_string_buffer(256)
    before = out.clone()
    rc = lib.md_energy_static(C.c_void_p(s.vel.data_ptr()), C.c_void_p(s.force.data_ptr()), None, api.ENERGY_STATIC_MAX_N + 1,
                              1.0, 0.0, C.c_void_p(out.data_ptr()), C.c_void_p(torch.cuda.current_stream().cuda_stream), err, 256)
    torch.cuda.synchronize()
    assert rc == -3 and b"MD_ENERGY_STATIC_MAX_N" in err.value            # MD_ERR_CAPACITY, with the limit in the message
    assert torch.equal(out, before)                                       # nothing was launched
    rc = lib.md_energy_static(C.c_void_p(s.vel.data_ptr()), C.c_void_p(s.force.data_ptr()), None, 0, 1.0, 0.0,
                              C.c_void_p(out.data_ptr()), None, err, 256)
    assert rc == -1 and err.value
    assert lib.md_energy_static(None, None, None, 1, 1.0, 0.0, None, None, None, 0) == -1   # NULL arrays, no message buffer
